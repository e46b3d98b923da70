// NUFFT Radon pair kernels for sm_100a (steps F1-F4 and B1-B4 of DESIGN.md).
//
// Fine-grid layout: cell (y, x) of group g holds P = 4 complex planes = 8 real slices in 32 bytes
// (one full DRAM sector): grid[((g G + y) G + x) P + p].  Plane p carries slice 8g+2p in its real part
// and slice 8g+2p+1 in its imaginary part: A is real-linear, so two real slices ride one complex
// transform (the Nyquist radial mode is excluded, reading G2, so nothing leaks between them).
// Every kernel below reads and writes whole 32-byte cells (or 16-byte halves of them).
#include <cstdlib>
#include "common.cuh"
#include "fft_line.cuh"

namespace tc {

__constant__ float c_kb[KB_DEG + 1];
void set_kb_coeffs(const float *h) { cudaMemcpyToSymbol(c_kb, h, sizeof(float) * (KB_DEG + 1)); }

long long &launch_counter() { static thread_local long long c = 0; return c; }

extern __shared__ float4 smem_f4[];

__device__ __forceinline__ int wrap(int i, int G) { return i < 0 ? i + G : (i >= G ? i - G : i); }

// ------------------------------------------------------------------------------------------------
// Line kernels: grid = (lines, groups); one CTA = one line of the 4 planes of a group; blockDim = 2 * slots
// (see fft_line.cuh).  E = 8 for lengths <= 4096 (1024 threads, <= 64 registers), 16 above.
#define TC_LB(E) __launch_bounds__((E) == 8 ? 1024 : 768)

// periodic index on the fine grid -> image index, or -1 in the zero padding
__device__ __forceinline__ int unpad(int x, int n, int G) { return x < n / 2 ? x + n / 2 : (x >= G - n / 2 ? x - (G - n / 2) : -1); }

// F1 + row FFT.  eq. (8) read backwards: g = f d(y_i) d(x_j), zero-padded to G at periodic index.
template <int E>
__global__ void TC_LB(E) k_fwd_rows(DevPlan d, const float *__restrict__ vol, int S, float2 *__restrict__ rowbuf) {
    float2 *sm = reinterpret_cast<float2 *>(smem_f4);
    const int i = blockIdx.x, g = blockIdx.y, n = d.n, G = d.G, pp = threadIdx.x & 1;
    const float di = d.deapod[i];
    const int s0 = 8 * g + 4 * pp;                            // this thread's 4 slices: s0 .. s0+3
    const float *v0 = vol + ((size_t)s0 * n + i) * n;
    const size_t ss = (size_t)n * n;
    float4 *out = reinterpret_cast<float4 *>(rowbuf) + ((size_t)g * n + i) * G * 2 + pp;
    fft_line<E>(sm, d.fG, d.twG, -1.f,
        [&](int x) {
            const int j = unpad(x, n, G);
            float4 r = make_float4(0.f, 0.f, 0.f, 0.f);
            if (j >= 0) {
                const float w = di * d.deapod[j];
                if (s0 < S) r.x = v0[j] * w;
                if (s0 + 1 < S) r.y = v0[ss + j] * w;
                if (s0 + 2 < S) r.z = v0[2 * ss + j] * w;
                if (s0 + 3 < S) r.w = v0[3 * ss + j] * w;
            }
            return r;
        },
        [&](int x, float4 v) { out[(size_t)x * 2] = v; });
}

// F2 column FFT; only the n non-zero rows are read.
template <int E>
__global__ void TC_LB(E) k_fwd_cols(DevPlan d, const float2 *__restrict__ rowbuf, float2 *__restrict__ grid) {
    float2 *sm = reinterpret_cast<float2 *>(smem_f4);
    const int x = blockIdx.x, g = blockIdx.y, n = d.n, G = d.G, pp = threadIdx.x & 1;
    const float4 *in = reinterpret_cast<const float4 *>(rowbuf) + ((size_t)g * n * G + x) * 2 + pp;
    float4 *out = reinterpret_cast<float4 *>(grid) + ((size_t)g * G * G + x) * 2 + pp;
    fft_line<E>(sm, d.fG, d.twG, -1.f,
        [&](int y) { const int i = unpad(y, n, G); return i >= 0 ? __ldg(&in[(size_t)i * G * 2]) : make_float4(0.f, 0.f, 0.f, 0.f); },
        [&](int y, float4 v) { out[(size_t)y * G * 2] = v; });
}

// B3 inverse column FFT (unnormalised, eq. (8)); only the n rows of the crop are written.
template <int E>
__global__ void TC_LB(E) k_adj_cols(DevPlan d, const float2 *__restrict__ grid, float2 *__restrict__ rowbuf) {
    float2 *sm = reinterpret_cast<float2 *>(smem_f4);
    const int x = blockIdx.x, g = blockIdx.y, n = d.n, G = d.G, pp = threadIdx.x & 1;
    const float4 *in = reinterpret_cast<const float4 *>(grid) + ((size_t)g * G * G + x) * 2 + pp;
    float4 *out = reinterpret_cast<float4 *>(rowbuf) + ((size_t)g * n * G + x) * 2 + pp;
    fft_line<E>(sm, d.fG, d.twG, +1.f,
        [&](int y) { return __ldg(&in[(size_t)y * G * 2]); },
        [&](int y, float4 v) { const int i = unpad(y, n, G); if (i >= 0) out[(size_t)i * G * 2] = v; });
}

// B3 inverse row FFT + B4 crop and deapodise ("division by phihat"); re -> slice 2p, im -> 2p+1.
template <int E>
__global__ void TC_LB(E) k_adj_rows(DevPlan d, const float2 *__restrict__ rowbuf, int S, float *__restrict__ vol) {
    float2 *sm = reinterpret_cast<float2 *>(smem_f4);
    const int i = blockIdx.x, g = blockIdx.y, n = d.n, G = d.G, pp = threadIdx.x & 1;
    const float4 *in = reinterpret_cast<const float4 *>(rowbuf) + ((size_t)g * n + i) * G * 2 + pp;
    const float di = d.deapod[i];
    const int s0 = 8 * g + 4 * pp;
    float *v0 = vol + ((size_t)s0 * n + i) * n;
    const size_t ss = (size_t)n * n;
    fft_line<E>(sm, d.fG, d.twG, +1.f,
        [&](int x) { return __ldg(&in[(size_t)x * 2]); },
        [&](int x, float4 v) {
            const int j = unpad(x, n, G);
            if (j >= 0) {
                const float w = di * d.deapod[j];
                if (s0 < S) v0[j] = v.x * w;
                if (s0 + 1 < S) v0[ss + j] = v.y * w;
                if (s0 + 2 < S) v0[2 * ss + j] = v.z * w;
                if (s0 + 3 < S) v0[3 * ss + j] = v.w * w;
            }
        });
}

#include "kernels_polar.inc"

}  // namespace tc
