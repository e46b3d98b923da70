// Shared-memory Stockham FFT for sm_100a: PC independent lines ("planes") of length n = 2^a 5^b per CTA.
//
// Each pass is an in-place autosort step: every thread first pulls all of its butterfly inputs
// into registers, the CTA synchronises, then the outputs go back to shared memory at the permuted
// positions.  Natural order in, natural order out, no digit reversal.  Shared-memory index i is
// stored at i + (i >> 4): one float2 of padding per 128 bytes keeps the power-of-two strides of the
// early passes off the same banks.
//
// Pass with radix R, stride s (product of earlier radices), l = n / s, m = l / R, butterfly b = (p, q),
// q = b mod s, p = b / s:   y[q + s (R p + k)] = w_l^{p k}  sum_j x[q + s (p + m j)] w_R^{j k}.
// Radix-5 passes go last so s is a power of two in every pass that has twiddles to look up.
#pragma once
#include <cuda_runtime.h>

namespace tc {

struct FftDesc {
    int n;          // length = first * 8^n8 * (five ? 5 : 1)
    int first;      // 0, 2 or 4: radix of the leading pass
    int n8;         // number of radix-8 passes
    int five;       // 1 if a trailing radix-5 pass
    int ps;         // padded plane stride in float2
};

__device__ __forceinline__ int pidx(int i) { return i + (i >> 4); }

__device__ __forceinline__ float2 cmul(float2 a, float2 b) {
    return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
// multiply by dir * i  (dir = -1: forward transform, e^{-2 pi i ...}; dir = +1: inverse)
__device__ __forceinline__ float2 cmuli(float2 a, float dir) { return make_float2(-dir * a.y, dir * a.x); }

template <int R> struct Bfly;

template <> struct Bfly<2> {
    __device__ static __forceinline__ void run(float2 (&v)[2], float) {
        float2 a = v[0], b = v[1];
        v[0] = cadd(a, b); v[1] = csub(a, b);
    }
};

template <> struct Bfly<4> {
    __device__ static __forceinline__ void run(float2 (&v)[4], float dir) {
        float2 t0 = cadd(v[0], v[2]), t1 = csub(v[0], v[2]);
        float2 t2 = cadd(v[1], v[3]), t3 = cmuli(csub(v[1], v[3]), dir);
        v[0] = cadd(t0, t2); v[2] = csub(t0, t2);
        v[1] = cadd(t1, t3); v[3] = csub(t1, t3);
    }
};

template <> struct Bfly<8> {
    __device__ static __forceinline__ void run(float2 (&v)[8], float dir) {
        const float h = 0.70710678118654752440f;
        float2 a[4], b[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) { a[j] = cadd(v[j], v[j + 4]); b[j] = csub(v[j], v[j + 4]); }
        // b_j *= w8^j,  w8 = e^{dir * 2 pi i / 8}
        b[1] = make_float2(h * (b[1].x - dir * b[1].y), h * (b[1].y + dir * b[1].x));
        b[2] = cmuli(b[2], dir);
        b[3] = make_float2(h * (-b[3].x - dir * b[3].y), h * (-b[3].y + dir * b[3].x));
        Bfly<4>::run(a, dir);
        Bfly<4>::run(b, dir);
#pragma unroll
        for (int k = 0; k < 4; ++k) { v[2 * k] = a[k]; v[2 * k + 1] = b[k]; }
    }
};

template <> struct Bfly<5> {
    __device__ static __forceinline__ void run(float2 (&v)[5], float dir) {
        const float c1 = 0.30901699437494742410f, c2 = -0.80901699437494742410f;   // cos(2pi/5), cos(4pi/5)
        const float s1 = 0.95105651629515357212f, s2 = 0.58778525229247312917f;    // sin(2pi/5), sin(4pi/5)
        float2 a1 = cadd(v[1], v[4]), a2 = cadd(v[2], v[3]);
        float2 d1 = csub(v[1], v[4]), d2 = csub(v[2], v[3]);
        float2 x0 = v[0];
        float2 e1 = make_float2(x0.x + c1 * a1.x + c2 * a2.x, x0.y + c1 * a1.y + c2 * a2.y);
        float2 e2 = make_float2(x0.x + c2 * a1.x + c1 * a2.x, x0.y + c2 * a1.y + c1 * a2.y);
        float2 f1 = cmuli(make_float2(s1 * d1.x + s2 * d2.x, s1 * d1.y + s2 * d2.y), dir);
        float2 f2 = cmuli(make_float2(s2 * d1.x - s1 * d2.x, s2 * d1.y - s1 * d2.y), dir);
        v[0] = make_float2(x0.x + a1.x + a2.x, x0.y + a1.y + a2.y);
        v[1] = cadd(e1, f1); v[4] = csub(e1, f1);
        v[2] = cadd(e2, f2); v[3] = csub(e2, f2);
    }
};

// One pass.  sm: PC planes of stride ps.  tw[i] = e^{-2 pi i * i / n} (forward sign), i in [0, n).
template <int R, int PC>
__device__ __forceinline__ void fft_pass(float2 *sm, int n, int ps, int log2s, const float2 *__restrict__ tw, float dir) {
    constexpr int MAXC = (32 + R * PC - 1) / (R * PC);
    const int nb = n / R;
    const int s = 1 << log2s;
    const int m = nb >> log2s;                 // l / R with l = n / s
    float2 v[MAXC][PC][R];
#pragma unroll
    for (int c = 0; c < MAXC; ++c) {
        int b = threadIdx.x + c * blockDim.x;
        if (b < nb) {
            int p = b >> log2s, q = b & (s - 1);
#pragma unroll
            for (int pl = 0; pl < PC; ++pl)
#pragma unroll
                for (int j = 0; j < R; ++j) v[c][pl][j] = sm[pl * ps + pidx(q + ((p + m * j) << log2s))];
        }
    }
    __syncthreads();
#pragma unroll
    for (int c = 0; c < MAXC; ++c) {
        int b = threadIdx.x + c * blockDim.x;
        if (b < nb) {
            int p = b >> log2s, q = b & (s - 1);
            float2 w[R];
            if (m > 1) {
                // w_l^{p k} = tw[p k s]; load k = 1, 2, 4 and build the rest by products
                int base = p << log2s;
                w[1] = __ldg(&tw[base]);
                if (R > 2) w[2] = __ldg(&tw[2 * base]);
                if (R > 3) w[3] = cmul(w[1], w[2]);
                if (R > 4) w[4] = __ldg(&tw[4 * base]);
                if (R > 5) { w[5] = cmul(w[4], w[1]); w[6] = cmul(w[4], w[2]); w[7] = cmul(w[4], w[3]); }
                if (dir > 0.f) {
#pragma unroll
                    for (int k = 1; k < R; ++k) w[k].y = -w[k].y;
                }
            }
#pragma unroll
            for (int pl = 0; pl < PC; ++pl) {
                Bfly<R>::run(v[c][pl], dir);
#pragma unroll
                for (int k = 0; k < R; ++k) {
                    float2 o = v[c][pl][k];
                    if (k > 0 && m > 1) o = cmul(o, w[k]);
                    sm[pl * ps + pidx(q + ((R * p + k) << log2s))] = o;
                }
            }
        }
    }
    __syncthreads();
}

// Whole transform; data must be in shared memory and visible (caller synchronised) before the call.
// blockDim.x must be >= PC * n / 32 (rounded up to a warp).  Pass order: one radix-2 or radix-4 pass
// (if log2 of the power-of-two part is not a multiple of 3), then radix-8 passes, then the radix-5 pass.
template <int PC>
__device__ __forceinline__ void fft_core(float2 *sm, const FftDesc &d, const float2 *__restrict__ tw, float dir) {
    int ls = 0;
    if (d.first == 2) { fft_pass<2, PC>(sm, d.n, d.ps, 0, tw, dir); ls = 1; }
    else if (d.first == 4) { fft_pass<4, PC>(sm, d.n, d.ps, 0, tw, dir); ls = 2; }
#pragma unroll 1
    for (int i = 0; i < d.n8; ++i, ls += 3) fft_pass<8, PC>(sm, d.n, d.ps, ls, tw, dir);
    if (d.five) fft_pass<5, PC>(sm, d.n, d.ps, ls, tw, dir);
}

}  // namespace tc
