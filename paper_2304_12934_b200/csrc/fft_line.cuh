// Line FFT with the first pass fused into the global load and the last pass fused into the global store.
//
// One CTA transforms one line of P = 4 complex planes, length n = 2^a 5^b.  Thread t owns plane pair
// pp = t & 1 (planes 2pp, 2pp+1 = one 16-byte half of a 32-byte cell) and butterfly slot bt = t >> 1, so the
// two lanes of a pair touch the two halves of the same cell in the same instruction: every global access is
// a whole sector.  Passes are Stockham autosort steps (see fft.cuh); only the passes in the middle go
// shared -> shared.  E = butterfly elements a thread holds per plane (8: one radix-8 butterfly).
//
//   first pass  (s = 1):  x[b + nb j] come from `ld(index)`;  y[R b + k] -> shared memory
//   middle passes:        shared -> registers -> (barrier) -> shared
//   last pass   (m = 1):  x[b + s j] from shared memory;  y[b + s k] go to `st(index, value)`
//
// ld(idx) returns float4 = (plane 2pp re, im, plane 2pp+1 re, im); st(idx, float4) stores the same.
#pragma once
#include "fft.cuh"

namespace tc {

struct LineCtx {
    float2 *sm;               // P planes of stride ps
    const float2 *tw;         // e^{-2 pi i k / n}
    int n, ps, pp, bt, nbt;   // nbt = butterfly slots = blockDim.x / 2
    float dir;
};

template <int R>
__device__ __forceinline__ void line_twiddles(const LineCtx &c, int base, float2 (&w)[R]) {
    w[1] = __ldg(&c.tw[base]);
    if (R > 2) w[2] = __ldg(&c.tw[2 * base]);
    if (R > 3) w[3] = cmul(w[1], w[2]);
    if (R > 4) w[4] = __ldg(&c.tw[4 * base]);
    if (R > 5) { w[5] = cmul(w[4], w[1]); w[6] = cmul(w[4], w[2]); w[7] = cmul(w[4], w[3]); }
    if (c.dir > 0.f) {
#pragma unroll
        for (int k = 1; k < R; ++k) w[k].y = -w[k].y;
    }
}

template <int R, int E, class LD>
__device__ __forceinline__ void line_first_pass(const LineCtx &c, LD ld) {
    constexpr int MAXC = (E + R - 1) / R;
    const int nb = c.n / R;
    float2 *s0 = c.sm + (2 * c.pp) * c.ps, *s1 = s0 + c.ps;
    float4 v[MAXC][R];
#pragma unroll
    for (int cc = 0; cc < MAXC; ++cc) {
        const int b = c.bt + cc * c.nbt;
        if (b < nb) {
#pragma unroll
            for (int j = 0; j < R; ++j) v[cc][j] = ld(b + nb * j);
        }
    }
#pragma unroll
    for (int cc = 0; cc < MAXC; ++cc) {
        const int b = c.bt + cc * c.nbt;
        if (b < nb) {
            float2 a0[R], a1[R], w[R];
#pragma unroll
            for (int j = 0; j < R; ++j) { a0[j] = make_float2(v[cc][j].x, v[cc][j].y); a1[j] = make_float2(v[cc][j].z, v[cc][j].w); }
            Bfly<R>::run(a0, c.dir); Bfly<R>::run(a1, c.dir);
            line_twiddles<R>(c, b, w);
#pragma unroll
            for (int k = 0; k < R; ++k) {
                const int o = pidx(R * b + k);
                s0[o] = k ? cmul(a0[k], w[k]) : a0[k];
                s1[o] = k ? cmul(a1[k], w[k]) : a1[k];
            }
        }
    }
    __syncthreads();
}

template <int R, int E>
__device__ __forceinline__ void line_mid_pass(const LineCtx &c, int log2s) {
    constexpr int MAXC = (E + R - 1) / R;
    const int nb = c.n / R, s = 1 << log2s, m = nb >> log2s;
    float2 *s0 = c.sm + (2 * c.pp) * c.ps, *s1 = s0 + c.ps;
    float2 a0[MAXC][R], a1[MAXC][R];
#pragma unroll
    for (int cc = 0; cc < MAXC; ++cc) {
        const int b = c.bt + cc * c.nbt;
        if (b < nb) {
            const int p = b >> log2s, q = b & (s - 1);
#pragma unroll
            for (int j = 0; j < R; ++j) {
                const int o = pidx(q + ((p + m * j) << log2s));
                a0[cc][j] = s0[o]; a1[cc][j] = s1[o];
            }
        }
    }
    __syncthreads();
#pragma unroll
    for (int cc = 0; cc < MAXC; ++cc) {
        const int b = c.bt + cc * c.nbt;
        if (b < nb) {
            const int p = b >> log2s, q = b & (s - 1);
            float2 w[R];
            Bfly<R>::run(a0[cc], c.dir); Bfly<R>::run(a1[cc], c.dir);
            line_twiddles<R>(c, p << log2s, w);
#pragma unroll
            for (int k = 0; k < R; ++k) {
                const int o = pidx(q + ((R * p + k) << log2s));
                s0[o] = k ? cmul(a0[cc][k], w[k]) : a0[cc][k];
                s1[o] = k ? cmul(a1[cc][k], w[k]) : a1[cc][k];
            }
        }
    }
    __syncthreads();
}

template <int R, int E, class ST>
__device__ __forceinline__ void line_last_pass(const LineCtx &c, ST st) {
    constexpr int MAXC = (E + R - 1) / R;
    const int s = c.n / R;                      // m = 1: p = 0, q = b
    const float2 *s0 = c.sm + (2 * c.pp) * c.ps, *s1 = s0 + c.ps;
#pragma unroll
    for (int cc = 0; cc < MAXC; ++cc) {
        const int b = c.bt + cc * c.nbt;
        if (b < s) {
            float2 a0[R], a1[R];
#pragma unroll
            for (int j = 0; j < R; ++j) { const int o = pidx(b + s * j); a0[j] = s0[o]; a1[j] = s1[o]; }
            Bfly<R>::run(a0, c.dir); Bfly<R>::run(a1, c.dir);
#pragma unroll
            for (int k = 0; k < R; ++k) st(b + s * k, make_float4(a0[k].x, a0[k].y, a1[k].x, a1[k].y));
        }
    }
}

__device__ __forceinline__ LineCtx line_ctx(float2 *sm, const FftDesc &d, const float2 *tw, float dir) {
    LineCtx c;
    c.sm = sm; c.tw = tw; c.n = d.n; c.ps = d.ps; c.pp = threadIdx.x & 1; c.bt = threadIdx.x >> 1; c.nbt = blockDim.x >> 1; c.dir = dir;
    return c;
}

// Passes after the first: radix-8 passes from stride 2^ls, then the fused last pass (radix 8, or 5 if d.five).
template <int E, class ST>
__device__ __forceinline__ void line_finish(const LineCtx &c, const FftDesc &d, int ls, int n8_left, ST st) {
    const int nmid = d.five ? n8_left : n8_left - 1;
#pragma unroll 1
    for (int i = 0; i < nmid; ++i, ls += 3) line_mid_pass<8, E>(c, ls);
    if (d.five) line_last_pass<5, E>(c, st);
    else line_last_pass<8, E>(c, st);
}

// global -> FFT -> global.  Needs at least two passes (n >= 16, not 2 or 4 alone).
template <int E, class LD, class ST>
__device__ __forceinline__ void fft_line(float2 *sm, const FftDesc &d, const float2 *tw, float dir, LD ld, ST st) {
    const LineCtx c = line_ctx(sm, d, tw, dir);
    if (d.first == 2) { line_first_pass<2, E>(c, ld); line_finish<E>(c, d, 1, d.n8, st); }
    else if (d.first == 4) { line_first_pass<4, E>(c, ld); line_finish<E>(c, d, 2, d.n8, st); }
    else { line_first_pass<8, E>(c, ld); line_finish<E>(c, d, 3, d.n8 - 1, st); }
}

// shared (already filled and synchronised) -> FFT -> global.
template <int E, class ST>
__device__ __forceinline__ void fft_line_from_smem(float2 *sm, const FftDesc &d, const float2 *tw, float dir, ST st) {
    const LineCtx c = line_ctx(sm, d, tw, dir);
    int ls = 0;
    if (d.first == 2) { line_mid_pass<2, E>(c, 0); ls = 1; }
    else if (d.first == 4) { line_mid_pass<4, E>(c, 0); ls = 2; }
    line_finish<E>(c, d, ls, d.n8, st);
}

}  // namespace tc
