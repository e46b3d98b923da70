// MBIR update kernels (steps M1-M4 of DESIGN.md): extrapolation, residual, qGGMRF prior stencil
// (eqs. (12)-(13); 26 neighbours P:L149), gradient step and the objective's reductions.
// Reductions accumulate in float64 and are deterministic: per-block partials, then one block adds them
// to the accumulator slot.  Accumulator layout: acc[0..15] results, acc[16 .. 16+RED_BLOCKS) scratch.
#include "common.cuh"

namespace tc {

constexpr int RED_BLOCKS = 1184;     // 148 SMs x 8
constexpr int RED_THREADS = 256;

__device__ __forceinline__ void block_reduce_to(double v, double *partials) {
    __shared__ double sh[RED_THREADS / 32];
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = v;
    __syncthreads();
    if (threadIdx.x < 32) {
        v = threadIdx.x < RED_THREADS / 32 ? sh[threadIdx.x] : 0.0;
        for (int o = 4; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
        if (threadIdx.x == 0) partials[blockIdx.x] = v;
    }
}

__global__ void k_final_reduce(const double *partials, int nb, double *acc, int slot, double scale) {
    __shared__ double sh[RED_THREADS];
    double v = 0.0;
    for (int i = threadIdx.x; i < nb; i += RED_THREADS) v += partials[i];
    sh[threadIdx.x] = v;
    __syncthreads();
    for (int o = RED_THREADS / 2; o > 0; o >>= 1) {
        if (threadIdx.x < o) sh[threadIdx.x] += sh[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) acc[slot] += scale * sh[0];
}

static void final_reduce(double *acc, int slot, double scale, cudaStream_t st) {
    k_final_reduce<<<1, RED_THREADS, 0, st>>>(acc + 16, RED_BLOCKS, acc, slot, scale);
    TC_COUNT_LAUNCH();
}

// ---- elementwise --------------------------------------------------------------------------------
__global__ void k_extrapolate(const float *__restrict__ x, const float *__restrict__ xm, float beta, float *__restrict__ y, size_t n) {
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const float a = x[i];
        y[i] = fmaf(beta, a - xm[i], a);
    }
}
__global__ void k_residual(const float *__restrict__ Ax, const float *__restrict__ Axm, const float *__restrict__ b, float beta,
                           float *__restrict__ Ay, float *__restrict__ r, size_t n) {
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const float a = Ax[i];
        const float ay = fmaf(beta, a - Axm[i], a);
        Ay[i] = ay;
        r[i] = ay - b[i];
    }
}
__global__ void k_candidate_sino(const float *__restrict__ Ay, const float *__restrict__ Ag, const float *__restrict__ b, float invL,
                                 float *__restrict__ Az, double *partials, size_t n) {
    double s = 0.0;
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const float az = fmaf(-invL, Ag[i], Ay[i]);
        Az[i] = az;
        const double e = (double)az - (double)b[i];
        s += e * e;
    }
    block_reduce_to(s, partials);
}
__global__ void k_sumsq(const float *__restrict__ v, size_t n, double *partials) {
    double s = 0.0;
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const double e = v[i];
        s += e * e;
    }
    block_reduce_to(s, partials);
}
__global__ void k_scale(float *v, float a, size_t n) {
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) v[i] *= a;
}

// ---- qGGMRF stencil -----------------------------------------------------------------------------
// h(D) = u^2 / (c + u^(2-p)), h'(D) = sign(D)/sigma * u (2c + p u^(2-p)) / (c + u^(2-p))^2, u = |D|/sigma.
struct PriorK { float inv_sigma, c, p, q; };     // q = 2 - p

__device__ __forceinline__ float upow(float u, float q) {                                       // u >= 0; 0 -> 0 (lg2 -> -inf, ex2 -> 0)
    float r;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(q * __log2f(u)));
    return r;
}

__device__ __forceinline__ float dh(float D, const PriorK &k) {
    const float u = fabsf(D) * k.inv_sigma;
    const float uq = upow(u, k.q);
    const float den = k.c + uq;
    const float v = __fdividef(k.inv_sigma * u * fmaf(k.p, uq, 2.f * k.c), den * den);     // MUFU.RCP + FMUL, 2 ulp
    return copysignf(v, D);
}
__device__ __forceinline__ float hval(float D, const PriorK &k) {
    const float u = fabsf(D) * k.inv_sigma;
    return __fdividef(u * u, k.c + upow(u, k.q));
}

// w_mn = (1/dist) / (6 + 12/sqrt2 + 8/sqrt3)  (reading G10)
#define TC_W_FACE 0.05234482976f
#define TC_W_EDGE 0.03701338413f
#define TC_W_CORN 0.03022130267f
__device__ __forceinline__ float wgt(int dz, int dy, int dx) {
    const int k = dz * dz + dy * dy + dx * dx;
    return k == 1 ? TC_W_FACE : (k == 2 ? TC_W_EDGE : TC_W_CORN);
}

// M2 + M3: g = atr + lambda grad H(y), z = y - g / L.  One thread per voxel, 32 x 8 tiles in-plane; the tile
// and its one-voxel halo for the three z-planes are staged in shared memory.
template <bool STEP>
__global__ void __launch_bounds__(256) k_prior_grad(const float *__restrict__ y, const float *atr, PriorK pk, float lambda,
                                                     float invL, float *g, float *__restrict__ z, int S, int n, int s_first) {
    __shared__ float t[3][10][34];
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    const int x0 = blockIdx.x * 32, y0 = blockIdx.y * 8, s = blockIdx.z + s_first;
    for (int e = threadIdx.x; e < 3 * 10 * 34; e += 256) {
        const int dz = e / 340, r = e % 340, yy = r / 34, xx = r % 34;
        const int gz = s + dz - 1, gy = y0 + yy - 1, gx = x0 + xx - 1;
        const bool in = gz >= 0 && gz < S && gy >= 0 && gy < n && gx >= 0 && gx < n;
        t[dz][yy][xx] = in ? y[((size_t)gz * n + gy) * n + gx] : __int_as_float(0x7fc00000);   // NaN marks "outside"
    }
    __syncthreads();
    const int gx = x0 + tx, gy = y0 + ty;
    if (gx >= n || gy >= n) return;
    const float c0 = t[1][ty + 1][tx + 1];
    float acc = 0.f;
#pragma unroll
    for (int dz = -1; dz <= 1; ++dz)
#pragma unroll
        for (int dy = -1; dy <= 1; ++dy)
#pragma unroll
            for (int dx = -1; dx <= 1; ++dx) {
                if (dz == 0 && dy == 0 && dx == 0) continue;
                const float v = t[dz + 1][ty + 1 + dy][tx + 1 + dx];
                if (v == v) acc = fmaf(wgt(dz, dy, dx), dh(c0 - v, pk), acc);     // neighbours outside the volume skipped (G12)
            }
    const size_t o = ((size_t)s * n + gy) * n + gx;
    const float gv = (atr ? atr[o] : 0.f) + lambda * acc;
    g[o] = gv;
    if (STEP) z[o] = fmaf(-invL, gv, c0);
}

// M4 prior term: H(z) = sum over unordered pairs, each counted once through its 13 "forward" offsets
// (dz = 0: right, and the three below; dz = +1: all nine).  Same 32 x 8 tile with a one-voxel halo as the gradient,
// two z-planes; owners are the first S_own slices (slabs: the slice above the core is only a neighbour).
__global__ void __launch_bounds__(256) k_prior_value(const float *__restrict__ zv, PriorK pk, double *partials, int S, int n, int S_own) {
    __shared__ float t[2][10][34];
    __shared__ double red[8];
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    const int ntx = (n + 31) / 32, nty = (n + 7) / 8;
    const long long ntiles = (long long)ntx * nty * S_own;
    double sum = 0.0;
    for (long long tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        const int s = (int)(tile / (ntx * nty)), r = (int)(tile % (ntx * nty));
        const int x0 = (r % ntx) * 32, y0 = (r / ntx) * 8;
        __syncthreads();
        for (int e = threadIdx.x; e < 2 * 10 * 34; e += 256) {
            const int dz = e / 340, q = e % 340, yy = q / 34, xx = q % 34;
            const int gz = s + dz, gy = y0 + yy - 1, gx = x0 + xx - 1;
            const bool in = gz < S && gy >= 0 && gy < n && gx >= 0 && gx < n;
            t[dz][yy][xx] = in ? zv[((size_t)gz * n + gy) * n + gx] : __int_as_float(0x7fc00000);   // NaN marks "outside"
        }
        __syncthreads();
        if (x0 + tx < n && y0 + ty < n) {
            const float c0 = t[0][ty + 1][tx + 1];
            float acc = 0.f;
#pragma unroll
            for (int dz = 0; dz <= 1; ++dz)
#pragma unroll
                for (int dy = -1; dy <= 1; ++dy)
#pragma unroll
                    for (int dx = -1; dx <= 1; ++dx) {
                        if (dz == 0 && (dy < 0 || (dy == 0 && dx <= 0))) continue;
                        const float v = t[dz][ty + 1 + dy][tx + 1 + dx];
                        if (v == v) acc = fmaf(wgt(dz, dy, dx), hval(c0 - v, pk), acc);
                    }
            sum += (double)acc;
        }
    }
    for (int o = 16; o > 0; o >>= 1) sum += __shfl_down_sync(0xffffffffu, sum, o);
    if (tx == 0) red[ty] = sum;
    __syncthreads();
    if (threadIdx.x == 0) {
        double v = 0.0;
        for (int k = 0; k < 8; ++k) v += red[k];
        partials[blockIdx.x] = v;
    }
}

// ---- wrappers -------------------------------------------------------------------------------------
static int ew_blocks(size_t n) { size_t b = (n + 255) / 256; return (int)(b < 148 * 16 ? (b ? b : 1) : 148 * 16); }
static PriorK mk(PriorDev pr) { PriorK k; k.inv_sigma = 1.f / pr.sigma; k.c = pr.c; k.p = pr.p; k.q = 2.f - pr.p; return k; }

void launch_extrapolate(const float *x, const float *xm, float beta, float *y, size_t n, cudaStream_t st) {
    k_extrapolate<<<ew_blocks(n), 256, 0, st>>>(x, xm, beta, y, n); TC_COUNT_LAUNCH();
}
void launch_residual(const float *Ax, const float *Axm, const float *b, float beta, float *Ay, float *r, size_t n, cudaStream_t st) {
    k_residual<<<ew_blocks(n), 256, 0, st>>>(Ax, Axm, b, beta, Ay, r, n); TC_COUNT_LAUNCH();
}
void launch_update(const float *y, const float *atr, PriorDev pr, float invL, float *g, float *z, int S, int n, cudaStream_t st,
                   int s_first, int n_out) {
    if (n_out < 0) n_out = S - s_first;
    dim3 gr((n + 31) / 32, (n + 7) / 8, n_out);
    if (z) k_prior_grad<true><<<gr, 256, 0, st>>>(y, atr, mk(pr), pr.lambda, invL, g, z, S, n, s_first);
    else   k_prior_grad<false><<<gr, 256, 0, st>>>(y, atr, mk(pr), pr.lambda, invL, g, nullptr, S, n, s_first);
    TC_COUNT_LAUNCH();
}
void launch_candidate_sino(const float *Ay, const float *Ag, const float *b, float invL, float *Az, double *acc, size_t n, cudaStream_t st) {
    k_candidate_sino<<<RED_BLOCKS, RED_THREADS, 0, st>>>(Ay, Ag, b, invL, Az, acc + 16, n); TC_COUNT_LAUNCH();
    final_reduce(acc, 0, 0.5, st);
}
void launch_prior(const float *z, PriorDev pr, float *grad, double *acc, int S, int n, cudaStream_t st, int S_own) {
    if (S_own < 0) S_own = S;
    if (grad) { PriorDev p1 = pr; p1.lambda = 1.f; launch_update(z, nullptr, p1, 0.f, grad, nullptr, S, n, st); }
    if (acc) {
        k_prior_value<<<RED_BLOCKS, RED_THREADS, 0, st>>>(z, mk(pr), acc + 16, S, n, S_own); TC_COUNT_LAUNCH();
        final_reduce(acc, 1, 1.0, st);
    }
}
void launch_sumsq(const float *v, size_t n, double *acc, int slot, cudaStream_t st) {
    k_sumsq<<<RED_BLOCKS, RED_THREADS, 0, st>>>(v, n, acc + 16); TC_COUNT_LAUNCH();
    final_reduce(acc, slot, 1.0, st);
}
void launch_scale(float *v, float a, size_t n, cudaStream_t st) {
    k_scale<<<ew_blocks(n), 256, 0, st>>>(v, a, n); TC_COUNT_LAUNCH();
}

}  // namespace tc
