// MBIR update kernels (steps M1-M4 of DESIGN.md): extrapolation, residual, qGGMRF prior stencil
// (eqs. (12)-(13); 26 neighbours P:L149), gradient step and the objective's reductions.
// Reductions accumulate in float64 and are deterministic: per-block partials, then one block adds them
// to the accumulator slot.  Accumulator layout: acc[0..15] results, acc[16 .. 16+RED_BLOCKS) scratch.
#include <cmath>
#include <algorithm>
#include "common.cuh"

namespace tc {

constexpr int RED_BLOCKS = 1184;     // 148 SMs x 8 (<= 2048: the partial-sum area acc[16 ..] holds two sets of 2048)
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

// scratch = which half of the partial-sum area (two reductions may run on two streams at once)
static void final_reduce(double *acc, int slot, double scale, cudaStream_t st, int scratch = 0) {
    k_final_reduce<<<1, RED_THREADS, 0, st>>>(acc + 16 + scratch * 2048, RED_BLOCKS, acc, slot, scale);
    TC_COUNT_LAUNCH();
}

// ---- elementwise --------------------------------------------------------------------------------
__global__ void k_extrapolate(const float *__restrict__ x, const float *__restrict__ xm, float beta, float *__restrict__ y, size_t n) {
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const float a = x[i];
        y[i] = fmaf(beta, a - xm[i], a);
    }
}
// r = A y - b with A y = A x + beta (A x - A x-) formed on the fly (M1: the extrapolated sinogram is never stored)
__global__ void k_residual(const float *__restrict__ Ax, const float *__restrict__ Axm, const float *__restrict__ b, float beta,
                           float *__restrict__ r, size_t n) {
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const float a = Ax[i];
        r[i] = fmaf(beta, a - Axm[i], a) - b[i];
    }
}
// Az = A y - alpha A g (A y from A0, A1 as above; A1 == nullptr: A0 is A y itself; Ag == nullptr: Az = A y) and the data term;
// optionally (rnext, only meaningful when A0 is A x) the next iteration's residual Az + beta_next (Az - A0) - b.
// No __restrict__: Az may alias any input (each thread reads its own elements before it writes them).
__global__ void k_candidate_sino(const float *A0, const float *A1, const float *Ag, const float *b, float beta, float alpha,
                                 float *Az, double *partials, size_t n, float *rnext, float beta_next) {
    double s = 0.0;
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const float a = A0[i];
        const float ay = A1 ? fmaf(beta, a - A1[i], a) : a;
        const float az = Ag ? fmaf(-alpha, Ag[i], ay) : ay;
        const float bi = b[i];
        Az[i] = az;
        // the residual of the NEXT iteration if this candidate is accepted (then A x = A z, A x- = A0): the expression of k_residual,
        // on values this thread holds anyway; rnext may alias Ag (read above)
        if (rnext) rnext[i] = fmaf(beta_next, az - a, az) - bi;
        const double e = (double)az - (double)bi;
        s += e * e;
    }
    block_reduce_to(s, partials);
}
// z = y - alpha g (projected on z >= 0 if nonneg), y = x + beta (x - x-): the candidate of the majorise-minimise step
__global__ void k_step(const float *__restrict__ x, const float *__restrict__ xm, float beta, const float *__restrict__ g, float alpha,
                       int nonneg, float *__restrict__ z, size_t n) {
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const float a = x[i];
        const float zc = fmaf(-alpha, g[i], fmaf(beta, a - xm[i], a));
        z[i] = nonneg ? fmaxf(zc, 0.f) : zc;
    }
}
__global__ void k_sumsq(const float *__restrict__ v, size_t n, double *partials) {
    double s = 0.0;
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const double e = v[i];
        s += e * e;
    }
    block_reduce_to(s, partials);
}
__global__ void k_dot_gzx(const float *__restrict__ g, const float *__restrict__ z, const float *__restrict__ x, size_t n, double *partials) {
    double s = 0.0;
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
        s += (double)g[i] * ((double)z[i] - (double)x[i]);
    block_reduce_to(s, partials);
}
// Beer-Lambert pre-pass + projection -> sinogram reorder: sino[s][a][u] = -log(max((I - dark) / (flat - dark), floor)),
// I = proj[a][s][u]; flat / dark are [s][u] (nullable: 1 / 0).  One thread per (a, s, u): both sides are contiguous along u.
__global__ void k_preprocess(const float *__restrict__ proj, const float *__restrict__ flat, const float *__restrict__ dark,
                             int na, int S, int nd, float floor_, float *__restrict__ sino) {
    const size_t n = (size_t)na * S * nd;
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const int u = (int)(i % nd);
        const size_t as = i / nd;
        const int s = (int)(as % S), a = (int)(as / S);
        const size_t su = (size_t)s * nd + u;
        const float dk = dark ? dark[su] : 0.f, fl = flat ? flat[su] : 1.f;
        const float t = fmaxf((proj[i] - dk) / (fl - dk), floor_);
        sino[((size_t)s * na + a) * nd + u] = -logf(t);
    }
}
__global__ void k_scale(float *v, float a, size_t n) {
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) v[i] *= a;
}

// ---- qGGMRF stencil -----------------------------------------------------------------------------
// h(D) = u^2 / (c + u^(2-p)), h'(D) = sign(D)/sigma * u (2c + p u^(2-p)) / (c + u^(2-p))^2, u = |D|/sigma.
struct PriorK { float inv_sigma, c, p, q; int nonneg; unsigned allow; float wscale; float k0, is2; };
// k0 = q lg2(1 / sigma): u^q = 2^(q lg2|D| + k0), one FFMA instead of two FMUL; is2 = 1 / sigma^2 (folded into the pair weights).
// q = 2 - p; nonneg: project the candidate on z >= 0; allow: which of the 13 forward offsets belong to the neighbour set (26: all;
// 10: the 8 in-plane neighbours and the two along z; 6: faces), wscale: renormalises the 1/distance weights to sum 1 over the set

// One evaluation = three MUFU (lg2, ex2, rcp), issued as the bare approximate instructions: u = 0 gives lg2 = -inf, ex2 = 0 (the
// right limit for q > 0; q = 0, i.e. p = 2, is selected away), and no range fix-ups or branches surround them.
__device__ __forceinline__ float lg2a(float x) { float r; asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float ex2a(float x) { float r; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float rcpa(float x) { float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float upowD(float D, const PriorK &k) { return k.q == 0.f ? 1.f : ex2a(fmaf(k.q, lg2a(fabsf(D)), k.k0)); }   // (|D| / sigma)^q

// The three evaluations below come WITHOUT the factor 1 / sigma^2: the callers multiply by W = w_mn / sigma^2 (one constant per offset class).
// h'(D) sigma^2 = D (2c + p u^q) / (c + u^q)^2   (h'(D) = sign(D)/sigma * u (...) / (...)^2 with u = |D|/sigma)
__device__ __forceinline__ float dh(float D, const PriorK &k) {
    const float uq = upowD(D, k);
    const float r = rcpa(k.c + uq);
    return (D * r) * (fmaf(k.p, uq, 2.f * k.c) * r);
}
// h(D) sigma^2 = D^2 / (c + u^q)
#ifndef TC_NO_RCP_NR
// reciprocal on the FMA pipe: magic-constant seed (12 %) and three Newton steps (4e-8); the value kernel is MUFU-bound (74 %):
// two MUFU per pair instead of three, 6.86 -> 6.56 ms per 128 slices of 2048^2 (the denominators c + u^q lie in [c, 1e30])
__device__ __forceinline__ float rcp_nr(float x) {
    float r = __int_as_float(0x7EF311C7 - __float_as_int(x));
    r = r * fmaf(-x, r, 2.f); r = r * fmaf(-x, r, 2.f); r = r * fmaf(-x, r, 2.f);
    return r;
}
__device__ __forceinline__ float hval(float D, const PriorK &k) { return D * D * rcp_nr(k.c + upowD(D, k)); }
#else
__device__ __forceinline__ float hval(float D, const PriorK &k) { return D * D * rcpa(k.c + upowD(D, k)); }
#endif
// h'(D) / D sigma^2 = (2c + p u^q) / (c + u^q)^2: the curvature of the quadratic surrogate of h at D (finite at D = 0: 2 / c)
__device__ __forceinline__ float hcurv(float D, const PriorK &k) {
    const float uq = upowD(D, k);
    const float r = rcpa(k.c + uq);
    return (fmaf(k.p, uq, 2.f * k.c) * r) * r;
}

// w_mn = (1/dist) / (6 + 12/sqrt2 + 8/sqrt3)  (reading G10)
#define TC_W_FACE 0.05234482976f
#define TC_W_EDGE 0.03701338413f
#define TC_W_CORN 0.03022130267f
__device__ __forceinline__ float wgt(int dz, int dy, int dx, float is2) {      // w_mn / sigma^2
    const int k = dz * dz + dy * dy + dx * dx;
    return (k == 1 ? TC_W_FACE : (k == 2 ? TC_W_EDGE : TC_W_CORN)) * is2;
}

// M2 + M3, pair-sharing form.  h' is odd, so the pair {m, n} gives +d to m and -d to n with d = w h'(y_m - y_n): every pair
// is evaluated ONCE (13 "forward" pairs per voxel instead of 26; the evaluation costs three MUFU and bounds the kernel).
// A CTA owns a 32 x PM_TY tile with a one-voxel halo ring (34 x (PM_TY + 2) threads, one per column; PM_TY = 12: 476 of 480) and marches
// through a chunk of slices: at slice s a thread evaluates its 4 in-plane forward pairs and its 9 pairs with slice s + 1,
// leaves d in shared memory for the partner (the in-plane ones are picked up in the same step, the 9 others in the next
// step), and the interior threads write g and z.  One warm-up step below the chunk supplies the first slice's incoming pairs.
constexpr int PM_ZC_MIN = 16, PM_ZC_MAX = 64;   // output slices per chunk: chosen per launch (pm_chunk)
#ifndef PM_TY
#define PM_TY 12
#endif
constexpr int PM_HY = PM_TY + 2, PM_LIVE = 34 * PM_HY;      // tile rows (PM_TY) plus the halo ring; threads that hold a column
constexpr int PM_THREADS = (PM_LIVE + 31) / 32 * 32;

// The input is y = x + beta (x - x-), formed while loading when xm != nullptr (M1 fused: y never reaches HBM in the in-core loop).
template <bool STEP, bool EXTRAP>
__global__ void __launch_bounds__(PM_THREADS) k_prior_grad_march(const float *__restrict__ y, const float *__restrict__ xm, float beta,
                                                                 const float *atr, PriorK pk, float lambda,
                                                                 float invL, float *g, float *__restrict__ z, int S, int n, int s_first, int n_out, int PM_ZC) {
    __shared__ float val[2][PM_HY][34];
    __shared__ float din[4][PM_HY][34];
    __shared__ float dup[2][9][PM_HY][34];
    const int t = threadIdx.x, hx = t % 34, hy = t / 34;
    const bool live = t < PM_LIVE;
    const int gx = blockIdx.x * 32 + hx - 1, gy = blockIdx.y * PM_TY + hy - 1;
    const bool inplane = live && gx >= 0 && gx < n && gy >= 0 && gy < n;
    const bool core = hx >= 1 && hx <= 32 && hy >= 1 && hy <= PM_TY;
    const bool interior = inplane && core;
    const int zlo = s_first + blockIdx.z * PM_ZC, zhi = min(zlo + PM_ZC, s_first + n_out);
    const int zstart = zlo > 0 ? zlo - 1 : 0;
    const float NaN = __int_as_float(0x7fc00000);
    const size_t plane = (size_t)n * n, pix = (size_t)gy * n + gx;
    // which of this thread's 13 forward pairs exist: partner inside the tile array, inside the image, and not a pair of two
    // halo voxels (those belong to other tiles).  Independent of z: computed once.
    unsigned mask = 0;
    {
        int o = 0;
        for (int dz = 0; dz <= 1; ++dz)
            for (int dy = -1; dy <= 1; ++dy)
                for (int dx = -1; dx <= 1; ++dx) {
                    if (dz == 0 && (dy < 0 || (dy == 0 && dx <= 0))) continue;
                    const int ny = hy + dy, nx = hx + dx, px = gx + dx, py = gy + dy;
                    const bool pcore = nx >= 1 && nx <= 32 && ny >= 1 && ny <= PM_TY;
                    if (inplane && ny >= 0 && ny < PM_HY && nx >= 0 && nx < 34 && px >= 0 && px < n && py >= 0 && py < n && (core || pcore)) mask |= 1u << o;
                    ++o;
                }
        mask &= pk.allow;
    }
    auto ldy = [&](size_t i) { const float a = y[i]; return EXTRAP ? fmaf(beta, a - xm[i], a) : a; };
    // values are fetched two slices ahead, so a load has a whole step to arrive; two barriers per step
    float c_cur = inplane ? ldy((size_t)zstart * plane + pix) : NaN;
    float c_nxt = (inplane && zstart + 1 < S) ? ldy((size_t)(zstart + 1) * plane + pix) : NaN;
    if (live) { val[zstart & 1][hy][hx] = c_cur; val[(zstart + 1) & 1][hy][hx] = c_nxt; }
    for (int zz = zstart; zz < zhi; ++zz) {
        const bool warm = zz < zlo;
        const float c_nn = (inplane && zz + 2 < S && zz + 1 < zhi) ? ldy((size_t)(zz + 2) * plane + pix) : NaN;
        __syncthreads();                 // values of zz, zz + 1 visible; everybody is done with the previous step's din / dup
        float acc = 0.f;
        if (live) {
            const unsigned mk = (warm ? mask & ~15u : mask) & (zz + 1 < S ? ~0u : 15u);     // no in-plane pairs in the warm-up step, no upward pairs at the top
            const float *vc = &val[zz & 1][hy][hx], *vu = &val[(zz + 1) & 1][hy][hx];
            int o = 0;
#pragma unroll
            for (int dy = 0; dy <= 1; ++dy)
#pragma unroll
                for (int dx = -1; dx <= 1; ++dx) {
                    if (dy == 0 && dx <= 0) continue;
                    const float ev = wgt(0, dy, dx, pk.is2) * dh(c_cur - vc[dy * 34 + dx], pk);       // evaluated unconditionally (a NaN halo is selected away)
                    const float dv = (mk >> o & 1) ? ev : 0.f;
                    din[o][hy][hx] = dv; acc += dv; ++o;
                }
#pragma unroll
            for (int dy = -1; dy <= 1; ++dy)
#pragma unroll
                for (int dx = -1; dx <= 1; ++dx) {
                    const float ev = wgt(1, dy, dx, pk.is2) * dh(c_cur - vu[dy * 34 + dx], pk);
                    const float dv = (mk >> o & 1) ? ev : 0.f;
                    dup[zz & 1][o - 4][hy][hx] = dv; acc += dv; ++o;
                }
        }
        __syncthreads();
        if (interior && !warm) {
            int o = 0;
#pragma unroll
            for (int dy = 0; dy <= 1; ++dy)
#pragma unroll
                for (int dx = -1; dx <= 1; ++dx) {
                    if (dy == 0 && dx <= 0) continue;
                    acc -= din[o][hy - dy][hx - dx]; ++o;
                }
            if (zz > zstart) {                                    // the pairs with the slice below (none at the bottom of the volume)
                o = 0;
#pragma unroll
                for (int dy = -1; dy <= 1; ++dy)
#pragma unroll
                    for (int dx = -1; dx <= 1; ++dx) { acc -= dup[(zz - 1) & 1][o][hy - dy][hx - dx]; ++o; }
            }
            const size_t oi = (size_t)zz * plane + pix;
            const float gvv = (atr ? atr[oi] : 0.f) + lambda * pk.wscale * acc;
            g[oi] = gvv;
            if (STEP) { const float zc = fmaf(-invL, gvv, c_cur); z[oi] = pk.nonneg ? fmaxf(zc, 0.f) : zc; }
        }
        c_cur = c_nxt; c_nxt = c_nn;
        if (live) val[zz & 1][hy][hx] = c_nn;       // slice zz + 2 replaces slice zz (read before the barrier above)
    }
}

// M4 prior term: H(z) = sum over unordered pairs, each counted once through its 13 "forward" offsets (dz = 0: right, and the
// three below; dz = +1: all nine).  The same tiles and chunks as k_prior_grad_march, every plane is loaded once; a pair is owned
// by its lower voxel, owners are the first S_own slices (slabs: the slice above the core is only a neighbour).  A fixed number of
// CTAs walks the (tile, chunk) items, so the float64 partial sums and their final order are deterministic.
// CURV = true: the curvature of the quadratic surrogate along a direction g instead (majorise-minimise step length):
//   sum over pairs of w h'(D)/D (g_m - g_n)^2,  D = y_m - y_n,  y = x + beta (x - x-) formed on load.
template <bool CURV>
__global__ void __launch_bounds__(PM_THREADS) k_prior_value_march(const float *__restrict__ zv, const float *__restrict__ xm, float beta,
                                                                  const float *__restrict__ gdir, PriorK pk, double *partials, int S, int n, int S_own, int PM_ZC) {
    __shared__ float val[2][PM_HY][34];
    __shared__ float gval[CURV ? 2 : 1][CURV ? PM_HY : 1][CURV ? 34 : 1];
    __shared__ double red[PM_THREADS / 32];
    const int t = threadIdx.x, hx = t % 34, hy = t / 34;
    const bool live = t < PM_LIVE;
    const bool core = hx >= 1 && hx <= 32 && hy >= 1 && hy <= PM_TY;
    const int ntx = (n + 31) / 32, nty = (n + PM_TY - 1) / PM_TY, nch = (S_own + PM_ZC - 1) / PM_ZC;
    const long long nitems = (long long)ntx * nty * nch;
    const size_t plane = (size_t)n * n;
    auto ldv = [&](size_t i) { const float a = zv[i]; return CURV ? fmaf(beta, a - xm[i], a) : a; };
    double sum = 0.0;
    for (long long item = blockIdx.x; item < nitems; item += gridDim.x) {
        const int ch = (int)(item / (ntx * nty)), r = (int)(item % (ntx * nty));
        const int gx = (r % ntx) * 32 + hx - 1, gy = (r / ntx) * PM_TY + hy - 1;
        const bool inplane = live && gx >= 0 && gx < n && gy >= 0 && gy < n;
        unsigned mask = 0;
        {
            int o = 0;
            for (int dz = 0; dz <= 1; ++dz)
                for (int dy = -1; dy <= 1; ++dy)
                    for (int dx = -1; dx <= 1; ++dx) {
                        if (dz == 0 && (dy < 0 || (dy == 0 && dx <= 0))) continue;
                        const int px = gx + dx, py = gy + dy;
                        if (inplane && core && px >= 0 && px < n && py >= 0 && py < n) mask |= 1u << o;
                        ++o;
                    }
            mask &= pk.allow;
        }
        const int zlo = ch * PM_ZC, zhi = min(zlo + PM_ZC, S_own);
        const size_t pix = (size_t)gy * n + gx;
        float c_cur = inplane ? ldv((size_t)zlo * plane + pix) : 0.f;
        float c_nxt = (inplane && zlo + 1 < S) ? ldv((size_t)(zlo + 1) * plane + pix) : 0.f;
        float g_cur = 0.f, g_nxt = 0.f;
        if (CURV) {
            g_cur = inplane ? gdir[(size_t)zlo * plane + pix] : 0.f;
            g_nxt = (inplane && zlo + 1 < S) ? gdir[(size_t)(zlo + 1) * plane + pix] : 0.f;
        }
        __syncthreads();                                    // the previous item's readers are done
        if (live) {
            val[zlo & 1][hy][hx] = c_cur; val[(zlo + 1) & 1][hy][hx] = c_nxt;
            if (CURV) { gval[zlo & 1][hy][hx] = g_cur; gval[(zlo + 1) & 1][hy][hx] = g_nxt; }
        }
        for (int zz = zlo; zz < zhi; ++zz) {
            const bool more = inplane && zz + 2 < S && zz + 1 < zhi;
            const float c_nn = more ? ldv((size_t)(zz + 2) * plane + pix) : 0.f;
            const float g_nn = (CURV && more) ? gdir[(size_t)(zz + 2) * plane + pix] : 0.f;
            __syncthreads();
            const unsigned mk = mask & (zz + 1 < S ? ~0u : 15u);
            if (mk) {
                const float *vc = &val[zz & 1][hy][hx], *vu = &val[(zz + 1) & 1][hy][hx];
                const float *gc = CURV ? &gval[zz & 1][hy][hx] : nullptr, *gu = CURV ? &gval[(zz + 1) & 1][hy][hx] : nullptr;
                float acc = 0.f;
                int o = 0;
#pragma unroll
                for (int dy = 0; dy <= 1; ++dy)
#pragma unroll
                    for (int dx = -1; dx <= 1; ++dx) {
                        if (dy == 0 && dx <= 0) continue;
                        {
                            float ev;
                            if (CURV) { const float dg = g_cur - gc[dy * 34 + dx]; ev = wgt(0, dy, dx, pk.is2) * hcurv(c_cur - vc[dy * 34 + dx], pk) * (dg * dg); }
                            else ev = wgt(0, dy, dx, pk.is2) * hval(c_cur - vc[dy * 34 + dx], pk);
                            acc += (mk >> o & 1) ? ev : 0.f;
                        }
                        ++o;
                    }
#pragma unroll
                for (int dy = -1; dy <= 1; ++dy)
#pragma unroll
                    for (int dx = -1; dx <= 1; ++dx) {
                        {
                            float ev;
                            if (CURV) { const float dg = g_cur - gu[dy * 34 + dx]; ev = wgt(1, dy, dx, pk.is2) * hcurv(c_cur - vu[dy * 34 + dx], pk) * (dg * dg); }
                            else ev = wgt(1, dy, dx, pk.is2) * hval(c_cur - vu[dy * 34 + dx], pk);
                            acc += (mk >> o & 1) ? ev : 0.f;
                        }
                        ++o;
                    }
                sum += (double)acc;
            }
            __syncthreads();
            c_cur = c_nxt; c_nxt = c_nn;
            if (live) val[zz & 1][hy][hx] = c_nn;
            if (CURV) { g_cur = g_nxt; g_nxt = g_nn; if (live) gval[zz & 1][hy][hx] = g_nn; }
        }
    }
    for (int o = 16; o > 0; o >>= 1) sum += __shfl_down_sync(0xffffffffu, sum, o);
    if ((t & 31) == 0) red[t >> 5] = sum;
    __syncthreads();
    if (t == 0) {
        double v = 0.0;
        for (int k = 0; k < PM_THREADS / 32; ++k) v += red[k];
        partials[blockIdx.x] = v * (double)pk.wscale;
    }
}

// ---- wrappers -------------------------------------------------------------------------------------
// A chunk starts with one warm-up slice step, so long chunks waste less (128 slices of 2048^2: MBIR iteration 33.5 ms with 16-slice
// chunks, 32.1 ms with 64); short ones keep small problems spread over the SMs: as long as tiles x chunks fill the machine.
static int pm_chunk(int n, int S) {
    const long long tiles = (long long)((n + 31) / 32) * ((n + PM_TY - 1) / PM_TY);
    const int nch_min = (int)((RED_BLOCKS + tiles - 1) / tiles);
    return std::max(PM_ZC_MIN, std::min(PM_ZC_MAX, S / std::max(nch_min, 1)));
}
static int ew_blocks(size_t n) { size_t b = (n + 255) / 256; return (int)(b < 148 * 16 ? (b ? b : 1) : 148 * 16); }
// forward-offset order of the march kernels: o = 0..3 in plane (dy, dx) = (0, 1), (1, -1), (1, 0), (1, 1); o = 4..12: dz = 1, (dy, dx) row-major
static PriorK mk(PriorDev pr) {
    PriorK k; k.inv_sigma = 1.f / pr.sigma; k.c = pr.c; k.p = pr.p; k.q = 2.f - pr.p; k.nonneg = pr.nonneg;
    k.k0 = (float)((2.0 - (double)pr.p) * std::log2(1.0 / (double)pr.sigma)); k.is2 = (float)(1.0 / ((double)pr.sigma * pr.sigma));
    const double s26 = 6.0 + 12.0 / std::sqrt(2.0) + 8.0 / std::sqrt(3.0);
    if (pr.nbr == 10) { k.allow = 0xFu | (1u << 8); k.wscale = (float)(s26 / (6.0 + 4.0 / std::sqrt(2.0))); }       // 8 in plane + 2 along z
    else if (pr.nbr == 6) { k.allow = (1u << 0) | (1u << 2) | (1u << 8); k.wscale = (float)(s26 / 6.0); }              // faces
    else { k.allow = 0x1FFFu; k.wscale = 1.f; }
    return k;
}

void launch_extrapolate(const float *x, const float *xm, float beta, float *y, size_t n, cudaStream_t st) {
    k_extrapolate<<<ew_blocks(n), 256, 0, st>>>(x, xm, beta, y, n); TC_COUNT_LAUNCH();
}
void launch_residual(const float *Ax, const float *Axm, const float *b, float beta, float *r, size_t n, cudaStream_t st) {
    k_residual<<<ew_blocks(n), 256, 0, st>>>(Ax, Axm, b, beta, r, n); TC_COUNT_LAUNCH();
}
void launch_update(const float *x, const float *xm, float beta, const float *atr, PriorDev pr, float invL, float *g, float *z, int S, int n,
                   cudaStream_t st, int s_first, int n_out) {
    if (n_out < 0) n_out = S - s_first;
    const int PM_ZC = pm_chunk(n, n_out);
    dim3 gr((n + 31) / 32, (n + PM_TY - 1) / PM_TY, (n_out + PM_ZC - 1) / PM_ZC);
    const PriorK k = mk(pr);
    if (xm) {
        if (z) k_prior_grad_march<true, true><<<gr, PM_THREADS, 0, st>>>(x, xm, beta, atr, k, pr.lambda, invL, g, z, S, n, s_first, n_out, PM_ZC);
        else   k_prior_grad_march<false, true><<<gr, PM_THREADS, 0, st>>>(x, xm, beta, atr, k, pr.lambda, invL, g, nullptr, S, n, s_first, n_out, PM_ZC);
    } else {
        if (z) k_prior_grad_march<true, false><<<gr, PM_THREADS, 0, st>>>(x, nullptr, 0.f, atr, k, pr.lambda, invL, g, z, S, n, s_first, n_out, PM_ZC);
        else   k_prior_grad_march<false, false><<<gr, PM_THREADS, 0, st>>>(x, nullptr, 0.f, atr, k, pr.lambda, invL, g, nullptr, S, n, s_first, n_out, PM_ZC);
    }
    TC_COUNT_LAUNCH();
}
void launch_step(const float *x, const float *xm, float beta, const float *g, float alpha, int nonneg, float *z, size_t n, cudaStream_t st) {
    k_step<<<ew_blocks(n), 256, 0, st>>>(x, xm, beta, g, alpha, nonneg, z, n); TC_COUNT_LAUNCH();
}
void launch_candidate_sino(const float *A0, const float *A1, const float *Ag, const float *b, float beta, float alpha, float *Az, double *acc,
                           size_t n, cudaStream_t st, float *rnext, float beta_next) {
    // second half of the partial-sum area: this reduction may run beside the prior's (launch_prior) on another stream
    k_candidate_sino<<<RED_BLOCKS, RED_THREADS, 0, st>>>(A0, A1, Ag, b, beta, alpha, Az, acc + 16 + 2048, n, rnext, beta_next); TC_COUNT_LAUNCH();
    final_reduce(acc, 0, 0.5, st, 1);
}
void launch_prior(const float *z, PriorDev pr, float *grad, double *acc, int S, int n, cudaStream_t st, int S_own) {
    if (S_own < 0) S_own = S;
    if (grad) { PriorDev p1 = pr; p1.lambda = 1.f; launch_update(z, nullptr, 0.f, nullptr, p1, 0.f, grad, nullptr, S, n, st); }
    if (acc) {
        k_prior_value_march<false><<<RED_BLOCKS, PM_THREADS, 0, st>>>(z, nullptr, 0.f, nullptr, mk(pr), acc + 16, S, n, S_own, pm_chunk(n, S_own)); TC_COUNT_LAUNCH();
        final_reduce(acc, 1, 1.0, st);
    }
}
void launch_prior_curvature(const float *x, const float *xm, float beta, const float *g, PriorDev pr, double *acc, int slot, int S, int n, cudaStream_t st) {
    k_prior_value_march<true><<<RED_BLOCKS, PM_THREADS, 0, st>>>(x, xm, beta, g, mk(pr), acc + 16, S, n, S, pm_chunk(n, S)); TC_COUNT_LAUNCH();
    final_reduce(acc, slot, 1.0, st);
}
void launch_sumsq(const float *v, size_t n, double *acc, int slot, cudaStream_t st) {
    k_sumsq<<<RED_BLOCKS, RED_THREADS, 0, st>>>(v, n, acc + 16); TC_COUNT_LAUNCH();
    final_reduce(acc, slot, 1.0, st);
}
void launch_dot_gzx(const float *g, const float *z, const float *x, size_t n, double *acc, int slot, cudaStream_t st) {
    k_dot_gzx<<<RED_BLOCKS, RED_THREADS, 0, st>>>(g, z, x, n, acc + 16); TC_COUNT_LAUNCH();
    final_reduce(acc, slot, 1.0, st);
}
void launch_preprocess(const float *proj, const float *flat, const float *dark, int na, int S, int nd, float floor_, float *sino, cudaStream_t st) {
    k_preprocess<<<ew_blocks((size_t)na * S * nd), 256, 0, st>>>(proj, flat, dark, na, S, nd, floor_, sino); TC_COUNT_LAUNCH();
}
void launch_scale(float *v, float a, size_t n, cudaStream_t st) {
    k_scale<<<ew_blocks(n), 256, 0, st>>>(v, a, n); TC_COUNT_LAUNCH();
}

}  // namespace tc
