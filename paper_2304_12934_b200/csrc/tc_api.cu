// C ABI of the tomoCAM B200 library (include/tc.h): plan, forward / adjoint pipelines, slab scheduler, MBIR loop.
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <chrono>
#include <string>
#include <vector>
#include <algorithm>
#include "../../include/tc.h"
#include "common.cuh"
#include <nvtx3/nvToolsExt.h>      // header-only NVTX: named ranges for Nsight timelines (stages, MBIR iterations); no-ops without a tool
#include <cub/device/device_scan.cuh>
#include <cub/device/device_radix_sort.cuh>

using namespace tc;

static thread_local std::string g_err;
static tc_status fail(tc_status s, const std::string &msg) { g_err = msg; return s; }
extern "C" const char *tc_last_error(void) { return g_err.c_str(); }
extern "C" long long tc_launch_count(int reset) { long long v = launch_counter(); if (reset) launch_counter() = 0; return v; }

#define CU(call)                                                                                   \
    do {                                                                                           \
        cudaError_t e_ = (call);                                                                   \
        if (e_ != cudaSuccess) {                                                                   \
            tc_status s_ = (e_ == cudaErrorMemoryAllocation) ? TC_ENOMEM : TC_ECUDA;               \
            return fail(s_, std::string(#call) + ": " + cudaGetErrorString(e_));                   \
        }                                                                                          \
    } while (0)
#define TCS(call) do { tc_status s_ = (call); if (s_ != TC_OK) return s_; } while (0)

struct tc_plan {
    tc_geom geom;
    std::vector<float> angles;
    DevPlan d;
    int max_slab;                 // slices per slab (multiple of 8), 0 = not yet decided
    // device tables
    float2 *twG = nullptr, *twD = nullptr, *ph_fwd = nullptr, *ph_adj = nullptr, *ph_fbp[4] = {nullptr, nullptr, nullptr, nullptr};
    int fbp_filter = -1;          // >= 0 only while tc_fbp runs: index into ph_fbp
    float *deapod = nullptr, *th_sorted = nullptr;
    double2 *cs = nullptr, *cs_sorted = nullptr;
    int *a_sorted = nullptr, *tile_nr = nullptr;
    TileRange *tile_rng = nullptr;
    unsigned *tap_offs = nullptr;
    int2 *taps = nullptr;
    unsigned *heavy = nullptr;
    long long n_taps = 0;
    unsigned *pair_offs = nullptr; int *pair_idx = nullptr; void *pair_w = nullptr;      // lists of the cell runs
    int *gt_tiles = nullptr; unsigned *gt_start = nullptr; int4 *gt_samples = nullptr;   // tile-binned gather tables
    float2 *static_scratch = nullptr;   // device address of g_static_scratch on the plan's device (tc_radon_static); null if the lookup failed
    bool gather_tiles = true;     // F3 as k_fwd_gather_tiles + k_fwd_radial (default) or as the fused ray-by-ray k_fwd_gather (TC_GATHER=ray)
    // scratch
    int ng_alloc = 0;
    float2 *rowbuf = nullptr, *grid = nullptr, *cpol = nullptr;
    double *acc = nullptr;        // 16 results + reduction scratch
    // host-pointer scheduler
    float *stage_in[2] = {nullptr, nullptr}, *stage_out[2] = {nullptr, nullptr};
    size_t stage_in_elems = 0, stage_out_elems = 0;
    cudaStream_t s_h2d = nullptr, s_comp = nullptr, s_d2h = nullptr;
    cudaStream_t s_aux = nullptr; cudaEvent_t ev_aux[2] = {nullptr, nullptr};   // MBIR: the data term of the objective beside the prior term
    tc_sched_stats stats{};
    // per-stage CUDA-event timing (tc_profile)
    bool prof = false, prof_open = false;
    struct ProfRec { int stage; cudaEvent_t a, b; };
    std::vector<ProfRec> prof_recs;
    std::vector<cudaEvent_t> prof_pool;
};

// Events are pooled and reused (no cudaEventCreate inside a timed loop); at most PROF_MAX_RECS records are kept between two
// tc_profile_read calls (a long tc_mbir run with profiling on then simply stops recording).
constexpr size_t PROF_MAX_RECS = 1 << 16;
static void prof_stage(tc_plan *p, int stage, cudaStream_t st, bool begin) {
    if (!p->prof) return;
    if (begin) {
        p->prof_open = false;
        if (p->prof_recs.size() >= PROF_MAX_RECS) return;
        tc_plan::ProfRec r; r.stage = stage;
        if (p->prof_pool.size() >= 2) {
            r.a = p->prof_pool.back(); p->prof_pool.pop_back();
            r.b = p->prof_pool.back(); p->prof_pool.pop_back();
        } else if (cudaEventCreate(&r.a) != cudaSuccess || cudaEventCreate(&r.b) != cudaSuccess) { cudaGetLastError(); return; }
        if (cudaEventRecord(r.a, st) != cudaSuccess) { cudaGetLastError(); p->prof_pool.push_back(r.a); p->prof_pool.push_back(r.b); return; }
        p->prof_recs.push_back(r);
        p->prof_open = true;
    } else if (p->prof_open) {
        if (cudaEventRecord(p->prof_recs.back().b, st) != cudaSuccess) {
            cudaGetLastError();
            p->prof_pool.push_back(p->prof_recs.back().a); p->prof_pool.push_back(p->prof_recs.back().b); p->prof_recs.pop_back();
        }
        p->prof_open = false;
    }
}
static const char *const STAGE_NAMES[TC_N_STAGES] = {"F1 fwd_rows", "F2 fwd_cols", "F3 fwd_gather", "B1 adj_radial", "B2 adj_spread", "B3 adj_cols", "B3+B4 adj_rows", "F4 fwd_radial"};
struct NvtxRange { explicit NvtxRange(const char *name) { nvtxRangePushA(name); } ~NvtxRange() { nvtxRangePop(); } };
#define STAGE(id, call) do { NvtxRange nv_(STAGE_NAMES[id]); prof_stage(p, id, st, true); call; prof_stage(p, id, st, false); } while (0)

// ---- scratch of the allocation-free forward projection (tc_radon_static) --------------------------------------------------------
// Callers that cannot call cudaMalloc (CUDA graph capture, tight serving loops, harnesses that forbid it) get ONE entry point whose
// FFT scratch is this file-scope array instead of the plan's lazily allocated buffers: fine grid, forward half-plane and polar
// coefficients of ONE group of 8 slices, for n <= 256 and n_angles * n_det <= 131072 (16 MiB, held by every GPU that loads the
// library until exit).  In host code the name `g_static_scratch` is a host-side stand-in, not a device address: the address is
// taken with cudaGetSymbolAddress here, at set-up, once per device, with that device current, and handed to the kernels as a pointer.
constexpr int TC_STATIC_MAX_N = 256;
constexpr size_t TC_STATIC_MAX_SAMPLES = 131072;                                          // n_angles * n_det
constexpr size_t TC_STATIC_GRID = (size_t)(2 * TC_STATIC_MAX_N) * (2 * TC_STATIC_MAX_N) * P;   // float2 elements: 8 MiB
constexpr size_t TC_STATIC_ROW = (size_t)TC_STATIC_MAX_N * (2 * TC_STATIC_MAX_N) * P;          // 4 MiB
constexpr size_t TC_STATIC_CPOL = TC_STATIC_MAX_SAMPLES * P;                                  // 4 MiB
static __device__ __align__(256) float2 g_static_scratch[TC_STATIC_GRID + TC_STATIC_ROW + TC_STATIC_CPOL];

static float2 *static_scratch_address() {
    constexpr int MAX_DEV = 64;
    static float2 *addr[MAX_DEV] = {nullptr};
    static bool tried[MAX_DEV] = {false};
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= MAX_DEV) { cudaGetLastError(); return nullptr; }
    if (!tried[dev]) {
        tried[dev] = true;
        void *q = nullptr;
        if (cudaGetSymbolAddress(&q, g_static_scratch) == cudaSuccess) addr[dev] = static_cast<float2 *>(q);
        else cudaGetLastError();                                     // tc_radon_static then fails with a clear error; nothing else uses it
    }
    return addr[dev];
}

// ---- host-side mathematics of the plan (float64) ---------------------------------------------------
static double bessel_i0(double x) {          // I0(x) = sum_k (x^2/4)^k / (k!)^2
    const double q = 0.25 * x * x;
    double term = 1.0, sum = 1.0;
    for (int k = 1; k < 200; ++k) { term *= q / ((double)k * k); sum += term; if (term < 1e-17 * sum) break; }
    return sum;
}
static double kb_beta(int W, double sigma) { return M_PI * std::sqrt((W / sigma) * (W / sigma) * (sigma - 0.5) * (sigma - 0.5) - 0.8); }

// phi as a function of z = 2 q - 1, q = 1 - (2 r / W)^2: Chebyshev interpolation, truncated, as monomials.
static void kb_poly(int W, double sigma, float *out) {
    const double beta = kb_beta(W, sigma), i0b = bessel_i0(beta);
    const int M = 64;
    std::vector<double> fz(M), zk(M);
    for (int k = 0; k < M; ++k) {
        zk[k] = std::cos(M_PI * (k + 0.5) / M);
        const double q = 0.5 * (zk[k] + 1.0);
        fz[k] = bessel_i0(beta * std::sqrt(q)) / i0b;
    }
    std::vector<double> cheb(KB_DEG + 1);
    for (int j = 0; j <= KB_DEG; ++j) {
        double s = 0.0;
        for (int k = 0; k < M; ++k) s += fz[k] * std::cos(j * M_PI * (k + 0.5) / M);
        cheb[j] = (j == 0 ? 1.0 : 2.0) * s / M;
    }
    // T_0 = 1, T_1 = z, T_{j+1} = 2 z T_j - T_{j-1}
    std::vector<std::vector<double>> T(KB_DEG + 1, std::vector<double>(KB_DEG + 1, 0.0));
    T[0][0] = 1.0; if (KB_DEG >= 1) T[1][1] = 1.0;
    for (int j = 1; j < KB_DEG; ++j)
        for (int k = 0; k <= KB_DEG; ++k) T[j + 1][k] = (k > 0 ? 2.0 * T[j][k - 1] : 0.0) - T[j - 1][k];
    for (int k = 0; k <= KB_DEG; ++k) {
        double s = 0.0;
        for (int j = 0; j <= KB_DEG; ++j) s += cheb[j] * T[j][k];
        out[k] = (float)s;
    }
}

// n = 2^a 3^b 5^c 7^d 17^e (a >= 1) as a pass list for the line engine: radix-16 passes first, then 8 / 4 / 2, then the odd
// factors 3, 7, 17 and 5 (one pass each; 5 last, as the compile-time list of n = 2560 has it); at most FFT_MAX_PASSES passes.
static bool make_fft_desc(int n, FftDesc &f) {
    int m = n, twos = 0, odd[4] = {0, 0, 0, 0};
    const int primes[4] = {3, 7, 17, 5};
    while (m % 2 == 0) { m /= 2; ++twos; }
    for (int q = 0; q < 4; ++q) while (m % primes[q] == 0) { m /= primes[q]; ++odd[q]; }
    if (m != 1 || twos < 1) return false;
    f.n = n; f.npass = 0;
    auto push = [&](int r) { if (f.npass >= FFT_MAX_PASSES) return false; f.radix[f.npass++] = r; return true; };
    while (twos >= 4) { if (!push(16)) return false; twos -= 4; }
    if (twos > 0 && !push(1 << twos)) return false;
    for (int q = 0; q < 4; ++q) for (int k = 0; k < odd[q]; ++k) if (!push(primes[q])) return false;
    if (f.npass < 2) {                              // 16 -> 4 x 4, 8 -> 4 x 2, 4 -> 2 x 2; 2 alone is not supported
        if (f.npass == 1 && f.radix[0] >= 4) { const int r = f.radix[0]; f.radix[0] = r == 4 ? 2 : 4; f.radix[1] = r / f.radix[0]; f.npass = 2; }
        else return false;
    }
    f.smem_cells = n + (n >> 4) + 1;
    return (size_t)f.smem_cells * 32 <= 227 * 1024 - 1024;
}

template <typename T> static cudaError_t upload(T **dst, const std::vector<T> &h) {
    cudaError_t e = cudaMalloc((void **)dst, h.size() * sizeof(T));
    if (e != cudaSuccess) return e;
    return cudaMemcpy(*dst, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice);
}

extern "C" tc_status tc_plan_create(const tc_geom *gm, int max_slab_slices, tc_plan **out) {
    if (!gm || !out) return fail(TC_EINVAL, "null argument");
    if (gm->n <= 0 || gm->n_det <= 0 || gm->n_angles <= 0 || !gm->angles) return fail(TC_EINVAL, "non-positive size or null angles");
    if ((gm->n & 1) || (gm->n_det & 1)) return fail(TC_EINVAL, "n and n_det must be even");
    for (int a = 0; a < gm->n_angles; ++a)
        if (!std::isfinite(gm->angles[a])) return fail(TC_EINVAL, "non-finite angle");
    if (gm->oversamp != 2.0f || (gm->kb_width != 4 && gm->kb_width != 6 && gm->kb_width != 8))
        return fail(TC_EUNSUPPORTED, "only oversamp = 2 and kb_width = 4, 6 or 8");
    if (gm->n % 32) return fail(TC_EUNSUPPORTED, "n must be a multiple of 32");
    tc_plan *p = new tc_plan();
    p->geom = *gm;
    p->angles.assign(gm->angles, gm->angles + gm->n_angles);
    p->geom.angles = p->angles.data();
    if (p->geom.center < 0) p->geom.center = 0.5f * gm->n_det;
    p->max_slab = max_slab_slices > 0 ? (max_slab_slices + 7) / 8 * 8 : 0;
    const int n = gm->n, nd = gm->n_det, na = gm->n_angles, G = 2 * n;
    DevPlan &d = p->d;
    d.n = n; d.nd = nd; d.na = na; d.G = G; d.sc = (double)G / nd;
    if (!make_fft_desc(n, d.fN) || !make_fft_desc(nd, d.fD)) { delete p; return fail(TC_EUNSUPPORTED, "n and n_det must be 2^a 3^b 5^c 7^d 17^e, a >= 1, with at most 5 FFT passes (and at most 6800)"); }
    if (nd / 2 - 1 > 0 && d.sc * (nd / 2 - 1) + 3 >= G / 2 + 3) { /* taps wrap at most once; always true for sc = G/nd */ }

    const int W = gm->kb_width; const double sigma = 2.0;
    d.W = W; d.hw = 0.5 * W; d.hwf = 0.5f * W; d.discR = G / 2 + W - 1;
    const double beta = kb_beta(W, sigma), i0b = bessel_i0(beta);
    kb_poly(W, sigma, d.kb);
    d.kbs = -8.f / (float)(W * W);
    set_fft_roots();
    std::vector<float> deapod(n);
    for (int j = 0; j < n; ++j) {
        const double x = j - n / 2, a = M_PI * W * x / G, s = std::sqrt(beta * beta - a * a);
        deapod[j] = (float)(i0b * s / (W * std::sinh(s)));
    }
    auto twiddles = [](int len) {
        std::vector<float2> t(len);
        for (int i = 0; i < len; ++i) { const double a = 2.0 * M_PI * i / len; t[i] = make_float2((float)std::cos(a), (float)-std::sin(a)); }
        return t;
    };
    std::vector<float2> phf(nd), pha(nd), phr(nd), phh(nd), phs(nd), phb(nd);   // forward / adjoint phases; adjoint x FBP weights (ramp, Hann, Shepp-Logan, Butterworth)
    const double centre = p->geom.center;
    for (int k = 0; k < nd; ++k) {
        const int m = k < nd / 2 ? k : k - nd;
        if (k == nd / 2) { phf[k] = pha[k] = phr[k] = phh[k] = phs[k] = phb[k] = make_float2(0.f, 0.f); continue; }
        const double a = 2.0 * M_PI * std::fmod((double)m * centre, (double)nd) / nd;
        phf[k] = make_float2((float)(std::cos(a) / nd), (float)(-std::sin(a) / nd));
        pha[k] = make_float2((float)(std::cos(a) / nd), (float)(std::sin(a) / nd));
        {   // eq. (4): |k| dk dtheta, the DC bin takes the mean of |k| over the bin
            const double ramp = (M_PI / na) * (m == 0 ? 0.25 / nd : std::fabs((double)m) / nd);
            const double hann = ramp * 0.5 * (1.0 + std::cos(2.0 * M_PI * m / nd));
            phr[k] = make_float2((float)(ramp * std::cos(a) / nd), (float)(ramp * std::sin(a) / nd));
            phh[k] = make_float2((float)(hann * std::cos(a) / nd), (float)(hann * std::sin(a) / nd));
            const double xs = M_PI * m / nd, shepp = ramp * (m == 0 ? 1.0 : std::sin(xs) / xs);           // filters of P:L68
            const double butter = ramp / (1.0 + std::pow(std::fabs((double)m) / (nd / 4.0), 4.0));
            phs[k] = make_float2((float)(shepp * std::cos(a) / nd), (float)(shepp * std::sin(a) / nd));
            phb[k] = make_float2((float)(butter * std::cos(a) / nd), (float)(butter * std::sin(a) / nd));
        }
    }
    std::vector<double2> cs(na), css(na);
    std::vector<float> ths(na);
    std::vector<int> order(na);
    std::vector<double> thm(na);
    for (int a = 0; a < na; ++a) {
        // the polar kernels work on the transposed (column-major) fine grid: swap the axes (exactly), theta' = pi/2 - theta
        const double th = 0.5 * M_PI - (double)p->angles[a];
        cs[a] = make_double2(d.sc * std::sin((double)p->angles[a]), d.sc * std::cos((double)p->angles[a]));
        double r = std::fmod(th, M_PI); if (r < 0) r += M_PI;
        thm[a] = r; order[a] = a;
    }
    std::sort(order.begin(), order.end(), [&](int a, int b) { return thm[a] < thm[b]; });
    for (int k = 0; k < na; ++k) { css[k] = cs[order[k]]; ths[k] = (float)thm[order[k]]; }
    cudaError_t e = cudaSuccess;
    auto twg = twiddles(G), twd = twiddles(nd);
    if (e == cudaSuccess) e = upload(&p->twG, twg);
    if (e == cudaSuccess) e = upload(&p->twD, twd);
    if (e == cudaSuccess) e = upload(&p->ph_fwd, phf);
    if (e == cudaSuccess) e = upload(&p->ph_adj, pha);
    if (e == cudaSuccess) e = upload(&p->ph_fbp[0], phr);
    if (e == cudaSuccess) e = upload(&p->ph_fbp[1], phh);
    if (e == cudaSuccess) e = upload(&p->ph_fbp[2], phs);
    if (e == cudaSuccess) e = upload(&p->ph_fbp[3], phb);
    if (e == cudaSuccess) e = upload(&p->deapod, deapod);
    if (e == cudaSuccess) e = upload(&p->cs, cs);
    if (e == cudaSuccess) e = upload(&p->cs_sorted, css);
    if (e == cudaSuccess) e = upload(&p->th_sorted, ths);
    if (e == cudaSuccess) e = upload(&p->a_sorted, order);
    if (e == cudaSuccess) e = cudaMalloc((void **)&p->acc, (16 + 4096) * sizeof(double));
    if (e != cudaSuccess) { tc_plan_destroy(p); return fail(e == cudaErrorMemoryAllocation ? TC_ENOMEM : TC_ECUDA, cudaGetErrorString(e)); }
    d.twG = p->twG; d.twD = p->twD; d.ph_fwd = p->ph_fwd; d.ph_adj = p->ph_adj; d.deapod = p->deapod;
    d.cs = p->cs; d.cs_sorted = p->cs_sorted; d.th_sorted = p->th_sorted; d.a_sorted = p->a_sorted;
    d.J = (int)std::floor(d.hw * std::sqrt(2.0) / d.sc + 0.5);
    {
        const int nt = ((G + 31) / 32) * ((G + 7) / 8);
        e = cudaMalloc((void **)&p->tile_rng, (size_t)nt * 4 * sizeof(TileRange));
        if (e == cudaSuccess) e = cudaMalloc((void **)&p->tile_nr, (size_t)nt * sizeof(int));
        if (e != cudaSuccess) { tc_plan_destroy(p); return fail(TC_ENOMEM, cudaGetErrorString(e)); }
        d.tile_rng = p->tile_rng; d.tile_nr = p->tile_nr;
        launch_tile_ranges(d, p->tile_rng, p->tile_nr, nullptr);
        e = cudaDeviceSynchronize();
        if (e != cudaSuccess) { tc_plan_destroy(p); return fail(TC_ECUDA, std::string("tile ranges: ") + cudaGetErrorString(e)); }
        // per-cell tap lists of the spread (B2): count, exclusive scan (cub), fill
        const size_t nc = (size_t)nt * 256;
        int *counts = nullptr; void *tmp = nullptr; size_t tmp_bytes = 0;
        e = cudaMalloc((void **)&counts, (nc + 1) * sizeof(int));
        if (e == cudaSuccess) e = cudaMalloc((void **)&p->tap_offs, (nc + 1) * sizeof(unsigned));
        if (e == cudaSuccess) e = cudaMemset(counts, 0, (nc + 1) * sizeof(int));
        if (e == cudaSuccess) {
            launch_spread_count(d, counts, nullptr);
            cub::DeviceScan::ExclusiveSum(nullptr, tmp_bytes, (const unsigned *)counts, p->tap_offs, (int)(nc + 1));
            e = cudaMalloc(&tmp, tmp_bytes);
        }
        if (e == cudaSuccess) e = cub::DeviceScan::ExclusiveSum(tmp, tmp_bytes, (const unsigned *)counts, p->tap_offs, (int)(nc + 1));
        unsigned total = 0;
        if (e == cudaSuccess) e = cudaMemcpy(&total, p->tap_offs + nc, sizeof(unsigned), cudaMemcpyDeviceToHost);
        cudaFree(counts); cudaFree(tmp);
        if (e == cudaSuccess) e = cudaMalloc((void **)&p->taps, (size_t)std::max(total, 1u) * sizeof(int2));
        if (e != cudaSuccess) { tc_plan_destroy(p); return fail(e == cudaErrorMemoryAllocation ? TC_ENOMEM : TC_ECUDA, std::string("spread tap lists: ") + cudaGetErrorString(e)); }
        p->n_taps = total;
        d.tap_offs = p->tap_offs; d.taps = p->taps;
        launch_spread_fill(d, nullptr);
        {   // cells with long lists: at most the disc of radius ~ 36 na / (2 pi SPREAD_HEAVY) cells; size the list for all cells with > SPREAD_HEAVY taps
            const size_t cap = std::min<size_t>(nc, (size_t)spread_run_cells() * ((size_t)total / SPREAD_HEAVY + 1));      // long lists and the cells of their runs
            unsigned *cnt = nullptr;
            e = cudaMalloc((void **)&p->heavy, cap * sizeof(unsigned));
            if (e == cudaSuccess) e = cudaMalloc((void **)&cnt, sizeof(unsigned));
            if (e == cudaSuccess) e = cudaMemset(cnt, 0, sizeof(unsigned));
            if (e == cudaSuccess) { launch_spread_heavy_list(d, (unsigned)nc, p->heavy, cnt, nullptr); e = cudaMemcpy(&d.n_heavy, cnt, sizeof(unsigned), cudaMemcpyDeviceToHost); }
            cudaFree(cnt);
            d.heavy = p->heavy;
            d.side = nullptr; d.ev_fork = d.ev_join = nullptr;
            if (e == cudaSuccess && d.n_heavy) {
                e = cudaStreamCreateWithFlags(&d.side, cudaStreamNonBlocking);
                if (e == cudaSuccess) e = cudaEventCreateWithFlags(&d.ev_fork, cudaEventDisableTiming);
                if (e == cudaSuccess) e = cudaEventCreateWithFlags(&d.ev_join, cudaEventDisableTiming);
            }
            if (e != cudaSuccess) { tc_plan_destroy(p); return fail(TC_ECUDA, std::string("spread heavy list: ") + cudaGetErrorString(e)); }
        }
        {   // lists of the cell pairs (k_adj_spread_pairs): count, exclusive scan, fill
            const size_t np = (size_t)nt * (256 / spread_run_cells());
            unsigned *pc = nullptr; void *tmp2 = nullptr; size_t tb2 = 0; unsigned ptotal = 0;
            d.pair_offs = nullptr; d.pair_idx = nullptr; d.pair_w = nullptr;
            e = cudaMalloc((void **)&pc, (np + 1) * sizeof(unsigned));
            if (e == cudaSuccess) e = cudaMemset(pc, 0, (np + 1) * sizeof(unsigned));
            if (e == cudaSuccess) e = cudaMalloc((void **)&p->pair_offs, (np + 1) * sizeof(unsigned));
            if (e == cudaSuccess) {
                launch_pair_count(d, pc, nullptr);
                cub::DeviceScan::ExclusiveSum(nullptr, tb2, pc, p->pair_offs, (int)(np + 1));
                e = cudaMalloc(&tmp2, tb2);
            }
            if (e == cudaSuccess) e = cub::DeviceScan::ExclusiveSum(tmp2, tb2, pc, p->pair_offs, (int)(np + 1));
            if (e == cudaSuccess) e = cudaMemcpy(&ptotal, p->pair_offs + np, sizeof(unsigned), cudaMemcpyDeviceToHost);
            cudaFree(pc); cudaFree(tmp2);
            if (e == cudaSuccess) e = cudaMalloc((void **)&p->pair_idx, (size_t)std::max(ptotal, 1u) * sizeof(int));
            if (e == cudaSuccess) e = cudaMalloc(&p->pair_w, (size_t)std::max(ptotal, 1u) * sizeof(float) * spread_run_cells());
            if (e != cudaSuccess) { tc_plan_destroy(p); return fail(e == cudaErrorMemoryAllocation ? TC_ENOMEM : TC_ECUDA, std::string("spread pair lists: ") + cudaGetErrorString(e)); }
            d.pair_offs = p->pair_offs;
            launch_pair_fill(d, p->pair_idx, p->pair_w, nullptr);
            d.pair_idx = p->pair_idx; d.pair_w = p->pair_w;
        }
        e = cudaDeviceSynchronize();
        if (e != cudaSuccess) { tc_plan_destroy(p); return fail(TC_ECUDA, std::string("spread tap lists: ") + cudaGetErrorString(e)); }
    }
    {   // tile-binned gather: samples sorted by tile (radix sort of (tile, sample) keys), tile offsets, tiles ordered by load
        const size_t ns = (size_t)na * nd;
        d.gt_ntx = gt_ntx(G, W); d.gt_nty = gt_nty(G, W);
        const int ntile = d.gt_ntx * d.gt_nty;
        unsigned long long *keys = nullptr, *keys2 = nullptr; void *tmp = nullptr; size_t tmp_bytes = 0; unsigned *counts = nullptr;
        const int end_bit = 32 + std::max(1, (int)std::ceil(std::log2((double)ntile + 1)));
        const unsigned nvalid = (unsigned)((size_t)na * (nd - 1));           // all but the Nyquist mode of every angle
        e = cudaMalloc((void **)&keys, ns * sizeof(unsigned long long));
        if (e == cudaSuccess) e = cudaMalloc((void **)&keys2, ns * sizeof(unsigned long long));
        if (e == cudaSuccess) e = cudaMalloc((void **)&counts, (size_t)ntile * sizeof(unsigned));
        if (e == cudaSuccess) e = cudaMemset(counts, 0, (size_t)ntile * sizeof(unsigned));
        if (e == cudaSuccess) e = cudaMalloc((void **)&p->gt_samples, (size_t)std::max(nvalid, 1u) * sizeof(int4));
        if (e == cudaSuccess) {
            launch_gt_keys(d, keys, nullptr);
            cub::DeviceRadixSort::SortKeys(nullptr, tmp_bytes, keys, keys2, (int)ns, 0, 64);
            e = cudaMalloc(&tmp, tmp_bytes);
        }
        if (e == cudaSuccess) e = cub::DeviceRadixSort::SortKeys(tmp, tmp_bytes, keys, keys2, (int)ns, 0, 64);
        (void)end_bit;
        if (e == cudaSuccess) { launch_gt_fill(d, keys2, nvalid, p->gt_samples, counts, nullptr); e = cudaDeviceSynchronize(); }
        std::vector<unsigned> hc(ntile), hs(ntile + 1, 0);
        if (e == cudaSuccess) e = cudaMemcpy(hc.data(), counts, (size_t)ntile * sizeof(unsigned), cudaMemcpyDeviceToHost);
        cudaFree(keys); cudaFree(keys2); cudaFree(tmp); cudaFree(counts);
        std::vector<int> live;
        if (e == cudaSuccess) {
            for (int t = 0; t < ntile; ++t) { hs[t + 1] = hs[t] + hc[t]; if (hc[t]) live.push_back(t); }
            std::stable_sort(live.begin(), live.end(), [&](int x, int y) { return hc[x] > hc[y]; });
            if (hs[ntile] != nvalid) { tc_plan_destroy(p); return fail(TC_ECUDA, "gather tiles: sample count mismatch"); }
            if (live.empty()) live.push_back(0);
            e = upload(&p->gt_tiles, live);
            if (e == cudaSuccess) e = upload(&p->gt_start, hs);
            // Order the samples of every tile so that the four samples a quarter-warp reads together (one 128-byte shared-memory
            // wavefront = four 32-byte cells) never share a bank group: a cell's bank group is (column >> 1) mod 4, the same for
            // every tap once the first tap's column is fixed modulo 8, so a quartet takes its samples from the four residues of one
            // parity (0, 2, 4, 6 or 1, 3, 5, 7).  Queues are filled in (angle, mode) order, so quartets stay close in cpol.
            std::vector<int4> hsmp(std::max(nvalid, 1u));
            if (e == cudaSuccess) e = cudaMemcpy(hsmp.data(), p->gt_samples, (size_t)nvalid * sizeof(int4), cudaMemcpyDeviceToHost);
            if (e == cudaSuccess) {
                std::vector<int4> bins[8], outv;
                for (int t = 0; t < ntile; ++t) {
                    if (!hc[t]) continue;
                    for (auto &b : bins) b.clear();
                    outv.clear();
                    for (unsigned i = hs[t]; i < hs[t + 1]; ++i) bins[hsmp[i].y & 7].push_back(hsmp[i]);
                    size_t head[8] = {0, 0, 0, 0, 0, 0, 0, 0};
                    for (int par = 0; par < 2; ++par)
                        for (;;) {
                            bool all = true;
                            for (int q = 0; q < 4; ++q) all = all && head[par + 2 * q] < bins[par + 2 * q].size();
                            if (!all) break;
                            for (int q = 0; q < 4; ++q) { outv.push_back(bins[par + 2 * q][head[par + 2 * q]]); ++head[par + 2 * q]; }
                        }
                    for (;;) {                                     // leftovers: up to four samples from the fullest queues with distinct bank groups
                        int pick[4] = {-1, -1, -1, -1}; bool any = false;
                        for (int q = 0; q < 4; ++q) {
                            size_t best = 0;
                            for (int par = 0; par < 2; ++par) { const int b = par + 2 * q; const size_t left = bins[b].size() - head[b]; if (left > best) { best = left; pick[q] = b; } }
                            any = any || pick[q] >= 0;
                        }
                        if (!any) break;
                        int placed = 0;
                        for (int q = 0; q < 4; ++q) if (pick[q] >= 0) { outv.push_back(bins[pick[q]][head[pick[q]]]); ++head[pick[q]]; ++placed; }
                        for (; placed < 4; ++placed) {             // fill the quartet from whatever is left (conflicts, rare)
                            int b = -1; size_t best = 0;
                            for (int k2 = 0; k2 < 8; ++k2) { const size_t left = bins[k2].size() - head[k2]; if (left > best) { best = left; b = k2; } }
                            if (b < 0) break;
                            outv.push_back(bins[b][head[b]]); ++head[b];
                        }
                    }
                    std::copy(outv.begin(), outv.end(), hsmp.begin() + hs[t]);
                }
                e = cudaMemcpy(p->gt_samples, hsmp.data(), (size_t)nvalid * sizeof(int4), cudaMemcpyHostToDevice);
            }
        }
        if (e != cudaSuccess) { tc_plan_destroy(p); return fail(e == cudaErrorMemoryAllocation ? TC_ENOMEM : TC_ECUDA, std::string("gather tiles: ") + cudaGetErrorString(e)); }
        d.gt_nlive = nvalid ? (int)live.size() : 0;
        {   // cut the crowded tiles into shorter group runs: a 16-group item should stay below ~5 % of one CTA's share of the samples
            const unsigned lim16 = std::max(64u, nvalid / (148u * 20u));
            d.gt_nh = d.gt_nm = 0;
            for (int r = 0; r < d.gt_nlive; ++r) {
                if (hc[live[r]] > 4 * lim16) d.gt_nh = r + 1;
                if (hc[live[r]] > lim16) d.gt_nm = r + 1;
            }
        }
        d.gt_tiles = p->gt_tiles; d.gt_start = p->gt_start; d.gt_samples = p->gt_samples;
        const char *env = std::getenv("TC_GATHER");
        p->gather_tiles = !(env && std::string(env) == "ray") || W != KB_W;      // the ray-by-ray kernel is built for W = 6 only
    }
    p->static_scratch = static_scratch_address();     // set-up: tc_radon_static itself makes no symbol lookup
    *out = p;
    return TC_OK;
}

static void free_scratch(tc_plan *p) {
    cudaFree(p->rowbuf); cudaFree(p->grid); cudaFree(p->cpol);
    p->rowbuf = p->grid = p->cpol = nullptr; p->ng_alloc = 0;
    for (int b = 0; b < 2; ++b) { cudaFree(p->stage_in[b]); cudaFree(p->stage_out[b]); p->stage_in[b] = p->stage_out[b] = nullptr; }
    p->stage_in_elems = p->stage_out_elems = 0;
}

extern "C" tc_status tc_plan_destroy(tc_plan *p) {
    if (!p) return TC_OK;
    free_scratch(p);
    cudaFree(p->twG); cudaFree(p->twD); cudaFree(p->ph_fwd); cudaFree(p->ph_adj); cudaFree(p->ph_fbp[0]); cudaFree(p->ph_fbp[1]); cudaFree(p->ph_fbp[2]); cudaFree(p->ph_fbp[3]); cudaFree(p->deapod);
    cudaFree(p->cs); cudaFree(p->cs_sorted); cudaFree(p->th_sorted); cudaFree(p->a_sorted); cudaFree(p->acc); cudaFree(p->tile_rng); cudaFree(p->tile_nr); cudaFree(p->tap_offs); cudaFree(p->taps); cudaFree(p->heavy); cudaFree(p->pair_offs); cudaFree(p->pair_idx); cudaFree(p->pair_w);
    cudaFree(p->gt_tiles); cudaFree(p->gt_start); cudaFree(p->gt_samples);
    if (p->d.side) cudaStreamDestroy(p->d.side);
    if (p->d.ev_fork) cudaEventDestroy(p->d.ev_fork);
    if (p->d.ev_join) cudaEventDestroy(p->d.ev_join);
    for (auto &r : p->prof_recs) { cudaEventDestroy(r.a); cudaEventDestroy(r.b); }
    for (auto &e : p->prof_pool) cudaEventDestroy(e);
    if (p->s_aux) cudaStreamDestroy(p->s_aux);
    for (auto &ev : p->ev_aux) if (ev) cudaEventDestroy(ev);
    if (p->s_h2d) cudaStreamDestroy(p->s_h2d);
    if (p->s_comp) cudaStreamDestroy(p->s_comp);
    if (p->s_d2h) cudaStreamDestroy(p->s_d2h);
    delete p;
    return TC_OK;
}

// bytes of scratch per group of 8 slices
static size_t group_bytes(const tc_plan *p) {
    const DevPlan &d = p->d;
    return ((size_t)d.G * d.G + (size_t)d.n * d.G + (size_t)d.na * d.nd) * P * sizeof(float2);
}

// Decide the slab size (slices per pass through the pipeline) and allocate scratch for it: at most `cap_groups` groups
// (0 = no cap) and at most `frac` of the free device memory.  Scratch only ever grows; a smaller request reuses what is there.
static tc_status ensure_scratch(tc_plan *p, int n_slices, int *slab_out, int cap_groups = 0, double frac = 0.45) {
    int want = (n_slices + 7) / 8;                                   // groups
    if (p->max_slab) want = std::min(want, p->max_slab / 8);
    if (cap_groups > 0) want = std::min(want, cap_groups);
    if (want > p->ng_alloc) {
        size_t fr = 0, tot = 0;
        CU(cudaMemGetInfo(&fr, &tot));
        const size_t have = (size_t)p->ng_alloc * group_bytes(p);
        const size_t budget = (size_t)((fr + have) * frac);
        const int fit = (int)std::max<size_t>(1, budget / group_bytes(p));
        want = std::min(want, fit);
    }
    if (want > p->ng_alloc) {
        cudaFree(p->rowbuf); cudaFree(p->grid); cudaFree(p->cpol);
        p->rowbuf = p->grid = p->cpol = nullptr; p->ng_alloc = 0;
        const DevPlan &d = p->d;
        CU(cudaMalloc((void **)&p->grid, (size_t)want * d.G * d.G * P * sizeof(float2)));
        CU(cudaMalloc((void **)&p->rowbuf, (size_t)want * d.n * d.G * P * sizeof(float2)));
        CU(cudaMalloc((void **)&p->cpol, (size_t)want * d.na * d.nd * P * sizeof(float2)));
        p->ng_alloc = want;
    }
    *slab_out = p->ng_alloc * 8;
    return TC_OK;
}

// ---- device pipelines (one slab, device pointers) ---------------------------------------------------
static void forward_slab(tc_plan *p, const float *vol, int S, float *sino, cudaStream_t st) {
    const int ng = (S + 7) / 8;
    STAGE(0, launch_fwd_rows(p->d, vol, S, ng, p->rowbuf, st));
    STAGE(1, launch_fwd_cols(p->d, p->rowbuf, ng, p->grid, st));
    if (p->gather_tiles) {
        STAGE(2, launch_fwd_gather_tiles(p->d, p->grid, ng, p->cpol, st));
        STAGE(7, launch_fwd_radial(p->d, p->cpol, S, ng, sino, st));
    } else {
        STAGE(2, launch_fwd_gather(p->d, p->grid, S, ng, sino, st));
    }
}
// B1-B4.  tc_fbp is the same pipeline with the FBP-weighted phase table in place of ph_adj (one multiply in B1): p->fbp_filter >= 0.
static void adjoint_slab(tc_plan *p, const float *sino, int S, float *vol, cudaStream_t st) {
    const int ng = (S + 7) / 8;
    DevPlan d1 = p->d;
    if (p->fbp_filter >= 0) d1.ph_adj = p->ph_fbp[p->fbp_filter];
    STAGE(3, launch_adj_radial(d1, sino, S, ng, p->cpol, st));
    STAGE(4, launch_adj_spread(p->d, p->cpol, ng, p->grid, st));
    STAGE(5, launch_adj_cols(p->d, p->grid, ng, p->rowbuf, st));
    STAGE(6, launch_adj_rows(p->d, p->rowbuf, S, ng, vol, st));
}

extern "C" tc_status tc_profile(tc_plan *p, int enable) {
    if (!p) return fail(TC_EINVAL, "null plan");
    p->prof = enable != 0;
    return TC_OK;
}
extern "C" tc_status tc_profile_read(tc_plan *p, double *ms, long long *launches) {
    if (!p || !ms || !launches) return fail(TC_EINVAL, "null argument");
    for (int i = 0; i < TC_N_STAGES; ++i) { ms[i] = 0.0; launches[i] = 0; }
    for (auto &r : p->prof_recs) {
        float t = 0.f;
        CU(cudaEventSynchronize(r.b));
        CU(cudaEventElapsedTime(&t, r.a, r.b));
        ms[r.stage] += t; launches[r.stage] += 1;
        p->prof_pool.push_back(r.a); p->prof_pool.push_back(r.b);
    }
    p->prof_recs.clear();
    return TC_OK;
}

extern "C" tc_status tc_host_alloc(size_t bytes, void **ptr) {
    if (!ptr || bytes == 0) return fail(TC_EINVAL, "bad argument");
    *ptr = nullptr;
    if (cudaMallocHost(ptr, bytes) != cudaSuccess) { cudaGetLastError(); *ptr = nullptr; return fail(TC_ENOMEM, "tc_host_alloc: pinned host memory"); }
    return TC_OK;
}
extern "C" tc_status tc_host_free(void *ptr) {
    if (ptr && cudaFreeHost(ptr) != cudaSuccess) { cudaGetLastError(); return fail(TC_EINVAL, "tc_host_free: not a tc_host_alloc pointer"); }
    return TC_OK;
}

static tc_status check_launch() {
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(TC_ECUDA, std::string("kernel launch: ") + cudaGetErrorString(e));
    return TC_OK;
}

static bool is_device_ptr(const void *ptr) {
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, ptr) != cudaSuccess) { cudaGetLastError(); return false; }
    return at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged;
}

// Owns device / pinned-host allocations and host registrations of one call: everything is released on every return path.
struct CallMem {
    std::vector<void *> dev, host, reg;
    template <class T> cudaError_t alloc(T **ptr, size_t elems) {
        cudaError_t e = cudaMalloc((void **)ptr, std::max<size_t>(elems, 1) * sizeof(T));
        if (e == cudaSuccess) dev.push_back(*ptr); else { *ptr = nullptr; cudaGetLastError(); }
        return e;
    }
    template <class T> cudaError_t alloc_host(T **ptr, size_t elems) {
        cudaError_t e = cudaMallocHost((void **)ptr, std::max<size_t>(elems, 1) * sizeof(T));
        if (e == cudaSuccess) host.push_back(*ptr); else { *ptr = nullptr; cudaGetLastError(); }
        return e;
    }
    // page-locks caller memory for the duration of the call if it is pageable; returns true if the range is pinned afterwards
    bool pin(const void *ptr, size_t bytes) {
        cudaPointerAttributes at;
        if (cudaPointerGetAttributes(&at, ptr) != cudaSuccess) { cudaGetLastError(); return false; }
        if (at.type == cudaMemoryTypeHost) return true;
        if (at.type != cudaMemoryTypeUnregistered) return false;
        if (cudaHostRegister(const_cast<void *>(ptr), bytes, cudaHostRegisterDefault) != cudaSuccess) { cudaGetLastError(); return false; }
        reg.push_back(const_cast<void *>(ptr));
        return true;
    }
    void release() {
        for (void *q : dev) cudaFree(q);
        for (void *q : host) cudaFreeHost(q);
        for (void *q : reg) cudaHostUnregister(q);
        dev.clear(); host.clear(); reg.clear();
    }
    ~CallMem() { release(); }
};

#include "tc_ops.cuh"
#include "tc_mbir_streamed.cuh"

// ---- allocation-free forward projection --------------------------------------------------------------------------------------------
// tc_radon for DEVICE pointers with the FFT scratch in g_static_scratch (above): no cudaMalloc, cudaFree or allocating library
// routine, whatever the plan has or has not allocated so far.  Slices go through in groups of 8, one after the other on `stream`.
// Nothing in the scratch has to start at zero (the half-plane and the polar coefficients are fully rewritten for every group, and
// the fine-grid cells the column kernel does not write are never used by the gather), so nothing is cleared; the array keeps the
// last call's contents.  EVERY call on a device shares the array: calls that overlap on the GPU (two streams, two plans, two host
// threads) race.
extern "C" tc_status tc_radon_static(tc_plan *p, const float *volume, int S, float *sinogram, void *stream) {
    if (!p || !volume || !sinogram) return fail(TC_EINVAL, "null argument");
    if (S <= 0) return fail(TC_EINVAL, "n_slices must be positive");
    const DevPlan &d = p->d;
    if (d.n > TC_STATIC_MAX_N || (size_t)d.na * d.nd > TC_STATIC_MAX_SAMPLES)
        return fail(TC_EUNSUPPORTED, "tc_radon_static: the static scratch holds n <= 256 and n_angles * n_det <= 131072 (this plan: n = " +
                                         std::to_string(d.n) + ", n_angles * n_det = " + std::to_string((size_t)d.na * d.nd) + "); use tc_radon");
    if (!p->static_scratch) return fail(TC_ECUDA, "tc_radon_static: cudaGetSymbolAddress of the static scratch failed at plan creation");
    if (!is_device_ptr(volume) || !is_device_ptr(sinogram)) return fail(TC_EINVAL, "tc_radon_static: device pointers only");
    float2 *grid = p->static_scratch, *rowbuf = grid + TC_STATIC_GRID, *cpol = rowbuf + TC_STATIC_ROW;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t vps = (size_t)d.n * d.n, sps = (size_t)d.na * d.nd;
    for (int s0 = 0; s0 < S; s0 += 8) {
        const int ns = std::min(8, S - s0);
        launch_fwd_rows(d, volume + (size_t)s0 * vps, ns, 1, rowbuf, st);
        launch_fwd_cols(d, rowbuf, 1, grid, st);
        launch_fwd_gather_tiles(d, grid, 1, cpol, st);
        launch_fwd_radial(d, cpol, ns, 1, sinogram + (size_t)s0 * sps, st);
    }
    return check_launch();
}
