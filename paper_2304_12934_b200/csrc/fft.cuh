// Register butterflies (radix 2, 4, 5, 8, 16) and the FFT descriptor of the line engine (fft_line.cuh).
//
// Bfly<R, INV>::run(v): v[k] <- sum_j v[j] e^{-+2 pi i j k / R}  (INV = false: forward sign "-", true: "+"),
// natural order in, natural order out.
#pragma once
#include <cuda_runtime.h>

namespace tc {

constexpr int FFT_MAX_PASSES = 5;

// n = radix[0] * ... * radix[npass-1]; radix-16 passes first, then the rest of the power of two, then the odd factors (3, 7, 17, 5); npass >= 2.
struct FftDesc {
    int n;
    int npass;
    int radix[FFT_MAX_PASSES];
    int smem_cells;     // padded cells of 4 planes (32 B) a line needs in shared memory
};

__device__ __forceinline__ float2 cmul(float2 a, float2 b) {
    return make_float2(fmaf(a.x, b.x, -a.y * b.y), fmaf(a.x, b.y, a.y * b.x));
}
__device__ __forceinline__ float2 cmulc(float2 a, float2 b) {       // a * conj(b)
    return make_float2(fmaf(a.x, b.x, a.y * b.y), fmaf(a.y, b.x, -a.x * b.y));
}
// Complex additions as packed FP32 pairs (FADD2 on sm_100): half the issue slots of the butterflies' additions; the line kernels
// are issue-bound once TMA feeds them (measured: step 16.78 -> 16.40 ms).  -DTC_NO_F32X2 restores the scalar form.
#ifndef TC_NO_F32X2
__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return __fadd2_rn(a, make_float2(-b.x, -b.y)); }
#else
__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
#endif
// multiply by -i (forward) or +i (inverse)
template <bool INV> __device__ __forceinline__ float2 crot(float2 a) { return INV ? make_float2(-a.y, a.x) : make_float2(a.y, -a.x); }
// multiply by (cos, -+sin) given as constants c, s > 0 meaning e^{-+ i phi}
template <bool INV> __device__ __forceinline__ float2 cmulk(float2 a, float c, float s) {
    return INV ? make_float2(fmaf(a.x, c, -a.y * s), fmaf(a.y, c, a.x * s)) : make_float2(fmaf(a.x, c, a.y * s), fmaf(a.y, c, -a.x * s));
}

template <bool INV> __device__ __forceinline__ void bfly4(float2 &a, float2 &b, float2 &c, float2 &d) {
    const float2 t0 = cadd(a, c), t1 = csub(a, c), t2 = cadd(b, d), t3 = crot<INV>(csub(b, d));
    a = cadd(t0, t2); c = csub(t0, t2);
    b = cadd(t1, t3); d = csub(t1, t3);
}

// Odd radices without a hand-written butterfly (3, 7, ...: detector sizes such as 2448 = 2^4 3^2 17): the plain DFT,
// R (R - 1) complex multiply-adds with the roots of unity from constant memory (immediate operands after unrolling).
constexpr int FFT_MAX_ODD = 17;
#ifdef TC_FFT_ROOTS_DEFINE
__constant__ float2 c_root[FFT_MAX_ODD + 1][FFT_MAX_ODD + 1];          // c_root[R][m] = e^{-2 pi i m / R}, odd R only (set_fft_roots)
#endif
template <int R, bool INV> struct Bfly {
#ifdef TC_FFT_ROOTS_DEFINE
    static_assert((R & 1) == 1 && R <= FFT_MAX_ODD, "generic butterfly: odd radices only");
    __device__ static __forceinline__ void run(float2 (&v)[R]) {
        float2 o[R];
#pragma unroll
        for (int k = 0; k < R; ++k) {
            float2 acc = v[0];
#pragma unroll
            for (int j = 1; j < R; ++j) {
                const float2 w = c_root[R][(j * k) % R];
                const float wy = INV ? -w.y : w.y;
                acc.x = fmaf(v[j].x, w.x, fmaf(-v[j].y, wy, acc.x));
                acc.y = fmaf(v[j].x, wy, fmaf(v[j].y, w.x, acc.y));
            }
            o[k] = acc;
        }
#pragma unroll
        for (int k = 0; k < R; ++k) v[k] = o[k];
    }
#endif
};

template <bool INV> struct Bfly<2, INV> {
    __device__ static __forceinline__ void run(float2 (&v)[2]) {
        const float2 a = v[0], b = v[1];
        v[0] = cadd(a, b); v[1] = csub(a, b);
    }
};

template <bool INV> struct Bfly<4, INV> {
    __device__ static __forceinline__ void run(float2 (&v)[4]) { bfly4<INV>(v[0], v[1], v[2], v[3]); }
};

template <bool INV> struct Bfly<8, INV> {
    __device__ static __forceinline__ void run(float2 (&v)[8]) {
        const float h = 0.70710678118654752440f;
        float2 a[4], b[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) { a[j] = cadd(v[j], v[j + 4]); b[j] = csub(v[j], v[j + 4]); }
        // b_j *= w8^j
        b[1] = INV ? make_float2(h * (b[1].x - b[1].y), h * (b[1].y + b[1].x)) : make_float2(h * (b[1].x + b[1].y), h * (b[1].y - b[1].x));
        b[2] = crot<INV>(b[2]);
        b[3] = INV ? make_float2(h * (-b[3].x - b[3].y), h * (b[3].x - b[3].y)) : make_float2(h * (b[3].y - b[3].x), h * (-b[3].y - b[3].x));
        bfly4<INV>(a[0], a[1], a[2], a[3]);
        bfly4<INV>(b[0], b[1], b[2], b[3]);
#pragma unroll
        for (int k = 0; k < 4; ++k) { v[2 * k] = a[k]; v[2 * k + 1] = b[k]; }
    }
};

template <bool INV> struct Bfly<5, INV> {
    __device__ static __forceinline__ void run(float2 (&v)[5]) {
        const float c1 = 0.30901699437494742410f, c2 = -0.80901699437494742410f;   // cos(2pi/5), cos(4pi/5)
        const float s1 = 0.95105651629515357212f, s2 = 0.58778525229247312917f;    // sin(2pi/5), sin(4pi/5)
        const float2 a1 = cadd(v[1], v[4]), a2 = cadd(v[2], v[3]);
        const float2 d1 = csub(v[1], v[4]), d2 = csub(v[2], v[3]);
        const float2 x0 = v[0];
        const float2 e1 = make_float2(x0.x + c1 * a1.x + c2 * a2.x, x0.y + c1 * a1.y + c2 * a2.y);
        const float2 e2 = make_float2(x0.x + c2 * a1.x + c1 * a2.x, x0.y + c2 * a1.y + c1 * a2.y);
        const float2 f1 = crot<INV>(make_float2(s1 * d1.x + s2 * d2.x, s1 * d1.y + s2 * d2.y));
        const float2 f2 = crot<INV>(make_float2(s2 * d1.x - s1 * d2.x, s2 * d1.y - s1 * d2.y));
        v[0] = make_float2(x0.x + a1.x + a2.x, x0.y + a1.y + a2.y);
        v[1] = cadd(e1, f1); v[4] = csub(e1, f1);
        v[2] = cadd(e2, f2); v[3] = csub(e2, f2);
    }
};

// 16 = 4 x 4: j = 4 j1 + j0, k = k0 + 4 k1, w16^{jk} = w4^{j1 k0} w16^{j0 k0} w4^{j0 k1}.
template <bool INV> struct Bfly<16, INV> {
    __device__ static __forceinline__ void run(float2 (&v)[16]) {
        const float c1 = 0.92387953251128675613f, s1 = 0.38268343236508977173f;   // cos, sin of pi/8
        const float h = 0.70710678118654752440f;
        // step 1: for each j0, radix 4 over j1: inputs v[j0 + 4 j1] -> A[j0][k0] kept in v[j0 + 4 k0]
#pragma unroll
        for (int j0 = 0; j0 < 4; ++j0) bfly4<INV>(v[j0], v[j0 + 4], v[j0 + 8], v[j0 + 12]);
        // step 2: A[j0][k0] *= w16^{j0 k0}
        v[5] = cmulk<INV>(v[5], c1, s1);                       // e = 1
        v[6] = cmulk<INV>(v[6], h, h);                         // e = 2
        v[7] = cmulk<INV>(v[7], s1, c1);                       // e = 3
        v[9] = cmulk<INV>(v[9], h, h);                         // e = 2
        v[10] = crot<INV>(v[10]);                              // e = 4
        v[11] = cmulk<INV>(v[11], -h, h);                      // e = 6
        v[13] = cmulk<INV>(v[13], s1, c1);                     // e = 3
        v[14] = cmulk<INV>(v[14], -h, h);                      // e = 6
        v[15] = cmulk<INV>(v[15], -c1, -s1);                   // e = 9
        // step 3: for each k0, radix 4 over j0: inputs v[j0 + 4 k0] -> y[k0 + 4 k1] ; results land in v[4 k0 + k1]
#pragma unroll
        for (int k0 = 0; k0 < 4; ++k0) bfly4<INV>(v[4 * k0], v[4 * k0 + 1], v[4 * k0 + 2], v[4 * k0 + 3]);
        // transpose 4 x 4 so that v[k0 + 4 k1] = y[k0 + 4 k1]
#pragma unroll
        for (int a = 0; a < 4; ++a)
#pragma unroll
            for (int b = a + 1; b < 4; ++b) { const float2 t = v[4 * a + b]; v[4 * a + b] = v[4 * b + a]; v[4 * b + a] = t; }
    }
};

}  // namespace tc
