// NUFFT Radon pair kernels for sm_100a (steps F1-F4 and B1-B4 of DESIGN.md).
//
// Fine-grid layout: cell (y, x) of group g holds P = 4 complex planes = 8 real slices in 32 bytes
// (one full DRAM sector): grid[((g G + y) G + x) P + p].  Plane p carries slice 8g+2p in its real part
// and slice 8g+2p+1 in its imaginary part: A is real-linear, so two real slices ride one complex
// transform (the Nyquist radial mode is excluded, reading G2, so nothing leaks between them).
// Every kernel below reads and writes whole 32-byte cells (or 16-byte halves of them).
#include <cstdlib>
#include "common.cuh"

namespace tc {

__constant__ float c_kb[KB_DEG + 1];
void set_kb_coeffs(const float *h) { cudaMemcpyToSymbol(c_kb, h, sizeof(float) * (KB_DEG + 1)); }

long long &launch_counter() { static thread_local long long c = 0; return c; }

extern __shared__ float4 smem_f4[];

__device__ __forceinline__ int wrap(int i, int G) { return i < 0 ? i + G : (i >= G ? i - G : i); }

// ------------------------------------------------------------------------------------------------
// F1 + row FFT.  grid = (n rows, ng * (P / PC)); CTA = one image row of PC planes.
// eq. (8) read backwards: g = f d(y_i) d(x_j), zero-padded to G at periodic index.
template <int PC>
__global__ void __launch_bounds__(512) k_fwd_rows(DevPlan d, const float *__restrict__ vol, int S, float2 *__restrict__ rowbuf) {
    float2 *sm = reinterpret_cast<float2 *>(smem_f4);
    const int i = blockIdx.x;
    const int g = blockIdx.y;
    const int n = d.n, G = d.G, ps = d.fG.ps;
    // with PC < P the CTA handles the 16-byte halves of its cells one after the other, so the pair meets in L2
    for (int h = 0; h < P / PC; ++h) {
        if (h) __syncthreads();
        const float di = d.deapod[i];
        // zero the padding region x in [n/2, G - n/2)
        for (int x = n / 2 + threadIdx.x; x < G - n / 2; x += blockDim.x)
#pragma unroll
            for (int pl = 0; pl < PC; ++pl) sm[pl * ps + pidx(x)] = make_float2(0.f, 0.f);
        for (int j = threadIdx.x; j < n; j += blockDim.x) {
            const float w = di * d.deapod[j];
            const int x = wrap(j - n / 2, G);
#pragma unroll
            for (int pl = 0; pl < PC; ++pl) {
                const int s0 = 8 * g + 2 * (h * PC + pl);
                float re = s0 < S ? vol[((size_t)s0 * n + i) * n + j] : 0.f;
                float im = s0 + 1 < S ? vol[((size_t)(s0 + 1) * n + i) * n + j] : 0.f;
                sm[pl * ps + pidx(x)] = make_float2(re * w, im * w);
            }
        }
        __syncthreads();
        fft_core<PC>(sm, d.fG, d.twG, -1.f);
        float4 *out = reinterpret_cast<float4 *>(rowbuf) + ((size_t)g * n + i) * G * 2;
        for (int t = threadIdx.x; t < G * (PC / 2); t += blockDim.x) {
            const int x = t / (PC / 2), hh = t % (PC / 2);
            float2 a = sm[(2 * hh) * ps + pidx(x)], b = sm[(2 * hh + 1) * ps + pidx(x)];
            out[(size_t)x * 2 + h * (PC / 2) + hh] = make_float4(a.x, a.y, b.x, b.y);
        }
    }
}

// F2 column FFT.  grid = (G columns, ng * (P / PC)).  Only the n non-zero rows are read.
template <int PC>
__global__ void __launch_bounds__(512) k_fwd_cols(DevPlan d, const float2 *__restrict__ rowbuf, float2 *__restrict__ grid) {
    float2 *sm = reinterpret_cast<float2 *>(smem_f4);
    const int x = blockIdx.x;
    const int g = blockIdx.y;
    const int n = d.n, G = d.G, ps = d.fG.ps;
    // with PC < P the CTA handles the 16-byte halves of its cells one after the other, so the pair meets in L2
    for (int h = 0; h < P / PC; ++h) {
        if (h) __syncthreads();
        for (int y = n / 2 + threadIdx.x; y < G - n / 2; y += blockDim.x)
#pragma unroll
            for (int pl = 0; pl < PC; ++pl) sm[pl * ps + pidx(y)] = make_float2(0.f, 0.f);
        const float4 *in = reinterpret_cast<const float4 *>(rowbuf) + ((size_t)g * n * G + x) * 2 + h * (PC / 2);
        for (int t = threadIdx.x; t < n * (PC / 2); t += blockDim.x) {
            const int i = t / (PC / 2), hh = t % (PC / 2);
            float4 v = __ldg(&in[(size_t)i * G * 2 + hh]);
            const int y = wrap(i - n / 2, G);
            sm[(2 * hh) * ps + pidx(y)] = make_float2(v.x, v.y);
            sm[(2 * hh + 1) * ps + pidx(y)] = make_float2(v.z, v.w);
        }
        __syncthreads();
        fft_core<PC>(sm, d.fG, d.twG, -1.f);
        float4 *out = reinterpret_cast<float4 *>(grid) + ((size_t)g * G * G + x) * 2 + h * (PC / 2);
        for (int t = threadIdx.x; t < G * (PC / 2); t += blockDim.x) {
            const int y = t / (PC / 2), hh = t % (PC / 2);
            float2 a = sm[(2 * hh) * ps + pidx(y)], b = sm[(2 * hh + 1) * ps + pidx(y)];
            out[(size_t)y * G * 2 + hh] = make_float4(a.x, a.y, b.x, b.y);
        }
    }
}

// B3 inverse column FFT (unnormalised, eq. (8)); only the n rows of the crop are written.
template <int PC>
__global__ void __launch_bounds__(512) k_adj_cols(DevPlan d, const float2 *__restrict__ grid, float2 *__restrict__ rowbuf) {
    float2 *sm = reinterpret_cast<float2 *>(smem_f4);
    const int x = blockIdx.x;
    const int g = blockIdx.y;
    const int n = d.n, G = d.G, ps = d.fG.ps;
    // with PC < P the CTA handles the 16-byte halves of its cells one after the other, so the pair meets in L2
    for (int h = 0; h < P / PC; ++h) {
        if (h) __syncthreads();
        const float4 *in = reinterpret_cast<const float4 *>(grid) + ((size_t)g * G * G + x) * 2 + h * (PC / 2);
        for (int t = threadIdx.x; t < G * (PC / 2); t += blockDim.x) {
            const int y = t / (PC / 2), hh = t % (PC / 2);
            float4 v = __ldg(&in[(size_t)y * G * 2 + hh]);
            sm[(2 * hh) * ps + pidx(y)] = make_float2(v.x, v.y);
            sm[(2 * hh + 1) * ps + pidx(y)] = make_float2(v.z, v.w);
        }
        __syncthreads();
        fft_core<PC>(sm, d.fG, d.twG, +1.f);
        float4 *out = reinterpret_cast<float4 *>(rowbuf) + ((size_t)g * n * G + x) * 2 + h * (PC / 2);
        for (int t = threadIdx.x; t < n * (PC / 2); t += blockDim.x) {
            const int i = t / (PC / 2), hh = t % (PC / 2);
            const int y = wrap(i - n / 2, G);
            float2 a = sm[(2 * hh) * ps + pidx(y)], b = sm[(2 * hh + 1) * ps + pidx(y)];
            out[(size_t)i * G * 2 + hh] = make_float4(a.x, a.y, b.x, b.y);
        }
    }
}

// B3 inverse row FFT + B4 crop and deapodise ("division by phihat"); re -> slice 2p, im -> 2p+1.
template <int PC>
__global__ void __launch_bounds__(512) k_adj_rows(DevPlan d, const float2 *__restrict__ rowbuf, int S, float *__restrict__ vol) {
    float2 *sm = reinterpret_cast<float2 *>(smem_f4);
    const int i = blockIdx.x;
    const int g = blockIdx.y;
    const int n = d.n, G = d.G, ps = d.fG.ps;
    // with PC < P the CTA handles the 16-byte halves of its cells one after the other, so the pair meets in L2
    for (int h = 0; h < P / PC; ++h) {
        if (h) __syncthreads();
        const float4 *in = reinterpret_cast<const float4 *>(rowbuf) + ((size_t)g * n + i) * G * 2;
        for (int t = threadIdx.x; t < G * (PC / 2); t += blockDim.x) {
            const int x = t / (PC / 2), hh = t % (PC / 2);
            float4 v = __ldg(&in[(size_t)x * 2 + h * (PC / 2) + hh]);
            sm[(2 * hh) * ps + pidx(x)] = make_float2(v.x, v.y);
            sm[(2 * hh + 1) * ps + pidx(x)] = make_float2(v.z, v.w);
        }
        __syncthreads();
        fft_core<PC>(sm, d.fG, d.twG, +1.f);
        const float di = d.deapod[i];
        for (int j = threadIdx.x; j < n; j += blockDim.x) {
            const float w = di * d.deapod[j];
            const int x = wrap(j - n / 2, G);
#pragma unroll
            for (int pl = 0; pl < PC; ++pl) {
                const int s0 = 8 * g + 2 * (h * PC + pl);
                float2 v = sm[pl * ps + pidx(x)];
                if (s0 < S) vol[((size_t)s0 * n + i) * n + j] = v.x * w;
                if (s0 + 1 < S) vol[((size_t)(s0 + 1) * n + i) * n + j] = v.y * w;
            }
        }
    }
}

#include "kernels_polar.inc"

}  // namespace tc
