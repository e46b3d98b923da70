// NUFFT Radon pair kernels for sm_100a (steps F1-F4 and B1-B4 of DESIGN.md).
//
// Fine-grid layout: cell (y, x) of group g holds P = 4 complex planes = 8 real slices in 32 bytes
// (one full DRAM sector): grid[((g G + y) G + x) P + p].  Plane p carries slice 8g+2p in its real part
// and slice 8g+2p+1 in its imaginary part: A is real-linear, so two real slices ride one complex
// transform (the Nyquist radial mode is excluded, reading G2, so nothing leaks between them).
// Every kernel below reads and writes whole 32-byte cells (or 16-byte halves of them).
#include <cstdlib>
#include <algorithm>
#include <string>
#include <cuda.h>          // CUtensorMap and its enums only: the encoder is fetched with cudaGetDriverEntryPoint, libcuda is not linked
#define TC_FFT_ROOTS_DEFINE       // this translation unit owns the constant table of the odd butterflies
#include "common.cuh"
#include "fft_line.cuh"

namespace tc {

void set_fft_roots() {
    static float2 h[FFT_MAX_ODD + 1][FFT_MAX_ODD + 1];
    for (int R = 1; R <= FFT_MAX_ODD; ++R)
        for (int m = 0; m <= FFT_MAX_ODD; ++m) {
            const double a = 2.0 * 3.14159265358979323846 * (m % R) / R;
            h[R][m] = make_float2((float)cos(a), (float)-sin(a));
        }
    cudaMemcpyToSymbol(c_root, h, sizeof(h));
}

long long &launch_counter() { static thread_local long long c = 0; return c; }

extern __shared__ float4 smem_f4[];

__device__ __forceinline__ int wrap(int i, int G) { return i < 0 ? i + G : (i >= G ? i - G : i); }

// ------------------------------------------------------------------------------------------------
// Line kernels: grid = (lines x CTAs per line, groups); one CTA = one line of PL of the 4 planes of a group (fft_line.cuh).
//
// Pruned split.  The fine grid has G = 2 n points per axis but only n of them carry data on the image side
// (zero padding, eq. (8)), so a length-G transform with n non-zero inputs is two length-n transforms:
//   Ghat[2 r + p] = sum_t h[t] mu_p(t) e^{-2 pi i r t / n},   p = 0, 1,   mu_p(t) = e^{-2 pi i p X(t) / G},
// where t < n runs over the image samples in wrapped order (t < n/2: image index t + n/2, periodic fine-grid
// index X = t; t >= n/2: image index t - n/2, X = t + n).  The adjoint direction is the transpose: two length-n
// inverse transforms of the even and odd inputs, the second multiplied by conj(mu_1) and added to the first.
// A line therefore needs n (not G) cells of shared memory (70 KB at n = 2048) and two 512-thread CTAs fit on an SM, so one
// CTA's loads overlap another's butterflies.
// Layouts (cells of P = 4 planes = 32 bytes): a sector-wide (32-byte) column access runs at 4.4 TB/s for loads but
// 2.8 TB/s for stores on B200 (measured), so every store stream below is contiguous and only two load streams
// are strided:
//   forward  rowbuf[g][i][x & 1][x >> 1]      rows written contiguously (F1), columns read with a row stride (F2)
//   grid     grid[g][x][y & 1][y >> 1]        column-major: F2 writes and B3 reads whole columns contiguously; the
//                                             polar kernels address single cells and do not care
//   adjoint  rowbuf[g][x][i]                  columns written contiguously (B3), rows read with a column stride (B3 rows)
#define TC_LB __launch_bounds__(Cfg::SLOTS * 4, 2)          // 4-plane CTAs (polar kernels): up to 512 threads
// row / column kernels: 4-plane CTAs (512 threads, two per SM) or 2-plane CTAs (256 threads, 35 KB of shared memory, four per SM;
// each CTA then touches 16-byte halves of the cells and the two CTAs of a line are launched next to each other)
#define TC_LB2 __launch_bounds__(Cfg::SLOTS * Cfg::PL, 8 / Cfg::PL)

template <class Cfg> __device__ __forceinline__ Cfg make_cfg(const FftDesc &f, int tws) {
    if constexpr (Cfg::is_static) return Cfg{};
    else { Cfg c; c.d = f; c.tws_ = tws; return c; }
}

// Only the disc of fine-grid cells within W/2 of some polar sample carries data: |kappa| < G/2, so cells with
// kx^2 + ky^2 > (G/2 + W - 1)^2 (21 % of the grid) are never read by the gather nor written by the spread; the column
// kernels neither store nor load them.  lim = discR^2 - kx^2 for the column at hand.
__device__ __forceinline__ int disc_limit(int x, int G, int R) { const int kx = x < G / 2 ? x : x - G; return R * R - kx * kx; }
__device__ __forceinline__ bool disc_live(int y, int G, int lim) { const int ky = y < G / 2 ? y : y - G; return ky * ky <= lim; }

struct Wrapped { int img, X; };      // image index and periodic fine-grid index of wrapped sample t (lo = t < n / 2)
__device__ __forceinline__ Wrapped wrapped(int t, int n, bool lo) { const int h = n >> 1; Wrapped w; w.img = lo ? t + h : t - h; w.X = lo ? t : t + n; return w; }

// F1 + row FFT.  eq. (8) read backwards: g = f d(y_i) d(x_j), zero-padded to G at periodic index.
template <class Cfg>
__global__ void TC_LB2 k_fwd_rows(DevPlan d, const float *__restrict__ vol, int S, float2 *__restrict__ rowbuf) {
    float2 *sm = reinterpret_cast<float2 *>(smem_f4);
    const Cfg cfg = make_cfg<Cfg>(d.fN, 2);
    constexpr int NH = 4 / Cfg::PL;                          // CTAs per line
    const int i = blockIdx.x / NH, g = blockIdx.y, n = cfg.n(), G = 2 * n, pl = Cfg::PL * (blockIdx.x % NH) + threadIdx.x % Cfg::PL;
    const float di = d.deapod[i];
    const int sre = 8 * g + 2 * pl;
    const bool hre = sre < S, him = sre + 1 < S;
    const float *vre = vol + ((size_t)sre * n + i) * n, *vim = vre + (size_t)n * n;
    float2 *out = rowbuf + ((size_t)g * n + i) * G * 4 + pl;
#pragma unroll 1
    for (int p = 0; p < 2; ++p) {
        fft_line<false>(sm, cfg, d.twG,
            [&](int t, bool lo) {
                const Wrapped w = wrapped(t, n, lo);
                const float sc = di * __ldg(&d.deapod[w.img]);
                float2 v = make_float2(hre ? __ldg(&vre[w.img]) * sc : 0.f, him ? __ldg(&vim[w.img]) * sc : 0.f);
                if (p) v = cmul(v, __ldg(&d.twG[w.X]));
                return v;
            },
            NoPre(), [&](int r, bool, float2 v, float2) { out[(size_t)(p * n + r) * 4] = v; });
        __syncthreads();
    }
}

// F2 column FFT; only the n non-zero rows exist in rowbuf.
template <class Cfg>
__global__ void TC_LB2 k_fwd_cols(DevPlan d, const float2 *__restrict__ rowbuf, float2 *__restrict__ grid) {
    float2 *sm = reinterpret_cast<float2 *>(smem_f4);
    const Cfg cfg = make_cfg<Cfg>(d.fN, 2);
    constexpr int NH = 4 / Cfg::PL;                          // CTAs per line
    const int x = blockIdx.x / NH, g = blockIdx.y, n = cfg.n(), G = 2 * n, pl = Cfg::PL * (blockIdx.x % NH) + threadIdx.x % Cfg::PL;
    const float2 *in = rowbuf + ((size_t)g * n * G + (size_t)(x & 1) * n + (x >> 1)) * 4 + pl;
    float2 *out = grid + ((size_t)g * G + x) * G * 4 + pl;
    const int lim = disc_limit(x, G, d.discR);
#pragma unroll 1
    for (int p = 0; p < 2; ++p) {
        fft_line<false>(sm, cfg, d.twG,
            [&](int t, bool lo) {
                const Wrapped w = wrapped(t, n, lo);
                float2 v = __ldg(&in[(size_t)w.img * G * 4]);
                if (p) v = cmul(v, __ldg(&d.twG[w.X]));
                return v;
            },
            NoPre(), [&](int r, bool, float2 v, float2) { if (disc_live(2 * r + p, G, lim)) out[(p * n + r) * 4] = v; });
        __syncthreads();
    }
}

// B3 inverse column FFT (unnormalised, eq. (8)); only the n rows of the crop are produced.
template <class Cfg>
__global__ void TC_LB2 k_adj_cols(DevPlan d, const float2 *__restrict__ grid, float2 *rowbuf) {
    float2 *sm = reinterpret_cast<float2 *>(smem_f4);
    const Cfg cfg = make_cfg<Cfg>(d.fN, 2);
    constexpr int NH = 4 / Cfg::PL;                          // CTAs per line
    const int x = blockIdx.x / NH, g = blockIdx.y, n = cfg.n(), G = 2 * n, pl = Cfg::PL * (blockIdx.x % NH) + threadIdx.x % Cfg::PL;
    const float2 *in = grid + ((size_t)g * G + x) * G * 4 + pl;
    float2 *out = rowbuf + ((size_t)g * G + x) * n * 4 + pl;                 // adjoint half-plane, column-major: [g][x][i]
    const int lim = disc_limit(x, G, d.discR);
#pragma unroll 1
    for (int p = 0; p < 2; ++p) {
        fft_line<true>(sm, cfg, d.twG,
            [&](int k, bool) { return disc_live(2 * k + p, G, lim) ? __ldg(&in[(p * n + k) * 4]) : make_float2(0.f, 0.f); },
            [&](int t, bool lo) { return p ? out[wrapped(t, n, lo).img * 4] : make_float2(0.f, 0.f); },   // this thread wrote it in phase 0
            [&](int t, bool lo, float2 v, float2 old) {
                const Wrapped w = wrapped(t, n, lo);
                if (p) { v = cmulc(v, __ldg(&d.twG[w.X])); v = cadd(v, old); }
                out[w.img * 4] = v;
            });
        __syncthreads();
    }
}

// B3 inverse row FFT + B4 crop and deapodise ("division by phihat"); re -> slice 2 pl, im -> 2 pl + 1.
template <class Cfg>
__global__ void TC_LB2 k_adj_rows(DevPlan d, const float2 *__restrict__ rowbuf, int S, float *vol) {
    float2 *sm = reinterpret_cast<float2 *>(smem_f4);
    const PlaneMajorLast<Cfg> cfg = make_cfg<PlaneMajorLast<Cfg>>(d.fN, 2);
    constexpr int NH = 4 / Cfg::PL;                          // CTAs per line
    const int i = blockIdx.x / NH, g = blockIdx.y, n = cfg.n(), G = 2 * n, pl = Cfg::PL * (blockIdx.x % NH) + threadIdx.x % Cfg::PL;
    const float2 *in = rowbuf + ((size_t)g * G * n + i) * 4 + pl;
    const float di = d.deapod[i];
    const int plo = Cfg::PL * (blockIdx.x % NH) + threadIdx.x / Cfg::SLOTS;     // plane of this thread in the (plane-major) last pass
    const int sre = 8 * g + 2 * plo;
    const bool hre = sre < S, him = sre + 1 < S;
    float *vre = vol + ((size_t)sre * n + i) * n, *vim = vre + (size_t)n * n;
#pragma unroll 1
    for (int p = 0; p < 2; ++p) {
        fft_line<true>(sm, cfg, d.twG,
            [&](int k, bool) { return __ldg(&in[(size_t)(2 * k + p) * n * 4]); },
            [&](int t, bool lo) {                                                   // this thread wrote them in phase 0
                const int j = wrapped(t, n, lo).img;
                return p ? make_float2(hre ? vre[j] : 0.f, him ? vim[j] : 0.f) : make_float2(0.f, 0.f);
            },
            [&](int t, bool lo, float2 v, float2 old) {
                const Wrapped w = wrapped(t, n, lo);
                const float sc = di * __ldg(&d.deapod[w.img]);
                if (p) v = cmulc(v, __ldg(&d.twG[w.X]));
                v.x = fmaf(v.x, sc, old.x); v.y = fmaf(v.y, sc, old.y);
                if (hre) vre[w.img] = v.x;
                if (him) vim[w.img] = v.y;
            });
        __syncthreads();
    }
}

// ---- test hooks: one complex plane in / out of the internal layouts (tc_stage_*, per-stage unit tests) ----------------------------
// nat[y][x] (row y <-> k_y, natural order) <-> plane `pl` of group 0 of the fine grid, grid[x][y & 1][y >> 1][P]
__global__ void k_grid_plane(float2 *grid, float2 *nat, int G, int pl, int put) {
    const size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x;
    if (i >= (size_t)G * G) return;
    const int y = (int)(i / G), x = (int)(i % G);
    float2 *cell = grid + (((size_t)x * G) + (size_t)(y & 1) * (G >> 1) + (y >> 1)) * 4 + pl;
    if (put) *cell = nat[i]; else nat[i] = *cell;
}
// nat[a][k] (k = m mod nd) <-> plane `pl` of group 0 of the polar coefficients, cpol[a][k][P]
__global__ void k_cpol_plane(float2 *cpol, float2 *nat, size_t n, int pl, int put) {
    const size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x;
    if (i >= n) return;
    if (put) cpol[i * 4 + pl] = nat[i]; else nat[i] = cpol[i * 4 + pl];
}
void launch_grid_plane(float2 *grid, float2 *nat, int G, int pl, bool put, cudaStream_t st) {
    k_grid_plane<<<(unsigned)(((size_t)G * G + 255) / 256), 256, 0, st>>>(grid, nat, G, pl, put ? 1 : 0);
}
void launch_cpol_plane(float2 *cpol, float2 *nat, size_t n, int pl, bool put, cudaStream_t st) {
    k_cpol_plane<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(cpol, nat, n, pl, put ? 1 : 0);
}

#include "kernels_polar.cuh"
#include "kernels_gather_tiles.cuh"
#include "kernels_line_tma.cuh"

}  // namespace tc
