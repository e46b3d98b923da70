// Included by kernels_nufft.cu inside namespace tc (after kernels_gather_tiles.cuh: mbarrier / bulk-copy primitives).
//
// Line kernels fed by the tensor-memory accelerator.  The plain line kernels (kernels_nufft.cu) bring a line in with ordinary
// loads inside the first butterfly pass, so all warps of a CTA sit through the DRAM latency of the line together and only the
// second CTA of the SM covers for them.  Here ONE persistent CTA per SM holds two groups of threads (named barriers), and the
// next line is brought into a raw shared-memory buffer by TMA (cp.async.bulk.tensor, completion on an mbarrier) while the groups
// run the passes of the current one: the strided 32-byte cells of a column are one 3-D tensor box per 256 rows, issued by one
// thread, and no warp ever waits for DRAM inside a pass.
//
// k_fwd_cols_tma (F2): the two groups are the two phases of the pruned split (even / odd outputs, kernels_nufft.cu) of the SAME
// column: they share the raw input (read from HBM once instead of once per phase) and own one work buffer each.
//   shared memory: raw [n cells] | work 0 | work 1 | mbarriers      (n = 2048: 64 KB + 2 x 68 KB; n = 1024: two CTAs per SM)

__device__ __forceinline__ void tma_load_3d(void *dst, const CUtensorMap *tm, int c0, int c1, int c2, unsigned long long *bar) {
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
                 ::"r"(smem_u32(dst)), "l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned long long *bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}

constexpr int LT_BOX_ROWS = 256;                                     // rows of one tensor box (the most a box dimension may have)
template <int N> struct LtSmem {
    static constexpr int RAW_BYTES = N * 32;
    static constexpr int WORK_CELLS = N + (N >> 4) + 1;              // = make_fft_desc's smem_cells
    static constexpr int WORK_BYTES = (WORK_CELLS * 32 + 127) / 128 * 128;
    static constexpr int TOTAL = RAW_BYTES + 2 * WORK_BYTES + 64;
};

template <class Cfg>
__global__ void __launch_bounds__(2 * Cfg::GROUP_THREADS, 1024 / (2 * Cfg::GROUP_THREADS)) k_fwd_cols_tma(DevPlan d, const __grid_constant__ CUtensorMap tm, int ng,
                                                                          float2 *__restrict__ grid) {
    extern __shared__ __align__(128) char lt_smem[];
    using SM = LtSmem<Cfg::n()>;
    const Cfg cfg{};
    constexpr int n = Cfg::n(), G = 2 * n, R0 = Cfg::radix(0);
    float2 *raw = reinterpret_cast<float2 *>(lt_smem);
    const int p = threadIdx.x / Cfg::GROUP_THREADS;                   // group = phase of the pruned split
    float2 *work = reinterpret_cast<float2 *>(lt_smem + SM::RAW_BYTES + p * SM::WORK_BYTES);
    unsigned long long *full = reinterpret_cast<unsigned long long *>(lt_smem + SM::RAW_BYTES + 2 * SM::WORK_BYTES), *empty = full + 1;
    if (threadIdx.x == 0) { mbar_init(full, 1); mbar_init(empty, 2); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    __syncthreads();
    const int nlines = G * ng;
    // lines in storage order of the half-plane (xs = (x & 1) n + (x >> 1)): the CTAs that run together read neighbouring sectors
    auto issue = [&](int line) {
        const int g = line / G, xs = line - g * G;
        mbar_arrive_expect_tx(full, SM::RAW_BYTES);
#pragma unroll
        for (int i = 0; i < n / LT_BOX_ROWS; ++i) tma_load_3d(lt_smem + i * LT_BOX_ROWS * 32, &tm, 0, xs, g * n + i * LT_BOX_ROWS, full);
    };
    if (threadIdx.x == 0 && (int)blockIdx.x < nlines) issue(blockIdx.x);
    const LineCtx c = line_ctx<Cfg>(work, d.twG);
    int k = 0;
    for (int line = blockIdx.x; line < nlines; line += gridDim.x, ++k) {
        const int g = line / G, xs = line - g * G, x = xs < n ? 2 * xs : 2 * (xs - n) + 1;
        float2 *out = grid + ((size_t)g * G + x) * G * 4 + c.pl;
        const int lim = disc_limit(x, G, d.discR);
        mbar_wait(full, k & 1);
        line_first<R0, false>(c, cfg, [&](int t, bool lo) {
            const Wrapped w = wrapped(t, n, lo);
            float2 v = raw[w.img * 4 + c.pl];
            if (p) v = cmul(v, __ldg(&d.twG[w.X]));
            return v;
        });
        // the group's barrier at the end of the first pass: nobody of this group reads raw any more
        if (line_tid<Cfg>() == 0) mbar_arrive(empty);
        if (threadIdx.x == 0 && line + (int)gridDim.x < nlines) {
            mbar_wait(empty, k & 1);
            fence_proxy_async();
            issue(line + gridDim.x);
        }
        static_finish<false, Cfg, 1, R0>(c, cfg, NoPre(), [&](int r, bool, float2 v, float2) { if (disc_live(2 * r + p, G, lim)) out[(p * n + r) * 4] = v; });
        line_sync<Cfg>();                                             // the last pass has read the work buffer
    }
}

// ---- host side: tensor map of the forward half-plane rowbuf[g][i][xs] as {8 floats, G, n ng} with boxes {8, 1, 256} ----------
typedef CUresult (*tc_encode_tiled_fn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                        const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                        CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
static tc_encode_tiled_fn tensor_map_encoder() {
    static tc_encode_tiled_fn fn = nullptr;
    static bool tried = false;
    if (!tried) {
        tried = true;
        void *f = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &f, cudaEnableDefault, &q) == cudaSuccess && q == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<tc_encode_tiled_fn>(f);
        else
            cudaGetLastError();
    }
    return fn;
}

static int lt_l2_promotion() {
    static int v = -1;
    if (v < 0) { const char *e = std::getenv("TC_TMA_L2"); v = e ? std::atoi(e) : 0; }
    return v;
}

// Pass list, group size and pipeline shape per line length (the lengths of BASELINE configs 3 and 4; others take the plain kernels)
template <int N, int TWS> struct LtSize;
template <int TWS> struct LtSize<2048, TWS> { using Cfg = Grouped<SCfg<4, 2048, TWS, 16, 16, 8>, 512>; static constexpr int NGRP = 2, NBUF = 3, CTAS = 1; };
template <int TWS> struct LtSize<1024, TWS> { using Cfg = Grouped<SCfg<4, 1024, TWS, 16, 16, 4>, 256>; static constexpr int NGRP = 4, NBUF = 6, CTAS = 2; };
static int lt_sm_count() {
    static int n_sm = 0;
    if (!n_sm) { int dev = 0; cudaGetDevice(&dev); cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev); if (n_sm <= 0) n_sm = 148; }
    return n_sm;
}
// tensor-map cache of one call site: re-encoded when the buffer or the number of groups changes
struct LtMapCache { const void *ptr = nullptr; int ng = 0, n = 0; CUtensorMap tm; };

// true if the TMA-fed kernel took the launch
template <int N>
static bool launch_fwd_cols_tma_n(const DevPlan &d, const float2 *rowbuf, int ng, float2 *grid, cudaStream_t st) {
    tc_encode_tiled_fn enc = tensor_map_encoder();
    if (!enc) return false;
    using Cfg = typename LtSize<N, 2>::Cfg;
    static thread_local LtMapCache c;          // per host thread: plans may be used from different threads (one plan, one thread at a time)
    if (c.ptr != rowbuf || c.ng != ng) {
        const cuuint64_t dims[3] = {8, (cuuint64_t)d.G, (cuuint64_t)d.n * ng};
        const cuuint64_t strides[2] = {32, (cuuint64_t)d.G * 32};
        const cuuint32_t box[3] = {8, 1, LT_BOX_ROWS}, es[3] = {1, 1, 1};
        const int l2 = lt_l2_promotion();
        const CUtensorMapL2promotion pr = l2 == 1 ? CU_TENSOR_MAP_L2_PROMOTION_L2_64B : l2 == 2 ? CU_TENSOR_MAP_L2_PROMOTION_L2_128B
                                        : l2 == 3 ? CU_TENSOR_MAP_L2_PROMOTION_L2_256B : CU_TENSOR_MAP_L2_PROMOTION_NONE;
        if (enc(&c.tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<float2 *>(rowbuf), dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                CU_TENSOR_MAP_SWIZZLE_NONE, pr, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS) { c.ptr = nullptr; return false; }
        c.ptr = rowbuf; c.ng = ng;
    }
    constexpr int sh = LtSmem<N>::TOTAL;
    static bool attr = false;
    if (!attr) { cudaFuncSetAttribute(k_fwd_cols_tma<Cfg>, cudaFuncAttributeMaxDynamicSharedMemorySize, sh); attr = true; }
    k_fwd_cols_tma<Cfg><<<std::min(LtSize<N, 2>::CTAS * lt_sm_count(), d.G * ng), 2 * Cfg::GROUP_THREADS, sh, st>>>(d, c.tm, ng, grid);
    TC_COUNT_LAUNCH();
    return true;
}
static bool launch_fwd_cols_tma(const DevPlan &d, const float2 *rowbuf, int ng, float2 *grid, cudaStream_t st) {
    switch (d.n) {
    case 2048: return launch_fwd_cols_tma_n<2048>(d, rowbuf, ng, grid, st);
    case 1024: return launch_fwd_cols_tma_n<1024>(d, rowbuf, ng, grid, st);
    default: return false;
    }
}

// ------------------------------------------------------------------------------------------------------------------------------
// Buffer-rotation pipeline for the other line kernels.  A task = one length-n transform of the 4 planes of one line (one phase of
// the pruned split).  NGRP groups of threads work on NGRP tasks at a time, each in its own shared-memory buffer; the remaining
// NBUF - NGRP buffers are being filled by TMA.  The raw line lands at the start of the buffer it will be transformed in
// (line_first_inplace), so a line needs one buffer, not two.  Task q of a CTA belongs to group q % NGRP and buffer q % NBUF:
//   j = q / NGRP, line slot m = q % NGRP + NGRP (j / NPH), phase = j % NPH   (the NPH phases of a line stay with one group, in order)
// and the group that finishes task q refills its buffer with task q + NBUF (one elected thread, after the group's barrier).
// Tasks past the end of the CTA's lines are "issued" as a plain arrival, so that every buffer's barrier sees every phase.
__device__ __forceinline__ void tma_load_4d(void *dst, const CUtensorMap *tm, int c0, int c1, int c2, int c3, unsigned long long *bar) {
    asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];"
                 ::"r"(smem_u32(dst)), "l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(smem_u32(bar)) : "memory");
}

template <int N, int NBUF> struct LpSmem {
    static constexpr int BUF_BYTES = ((N + (N >> 4) + 1) * 32 + 127) / 128 * 128;
    static constexpr int TOTAL = NBUF * BUF_BYTES + 128;
};

struct LpTask { int m, phase; bool valid; };

// ISSUE(q, task, buffer, barrier): called by ONE thread; must arrive once on the barrier (arrive.expect_tx + copies, or plain arrive)
// WORK(task, buffer): called by all threads of the task's group once the buffer is full; ends with the group's barrier
template <class Cfg, int NGRP, int NBUF, int NPH, class ISSUE, class WORK>
__device__ __forceinline__ void line_pipeline(char *smem, int M, ISSUE issue, WORK work) {
    using SM = LpSmem<Cfg::n(), NBUF>;
    unsigned long long *full = reinterpret_cast<unsigned long long *>(smem + NBUF * SM::BUF_BYTES);
    if (threadIdx.x == 0)
        for (int b = 0; b < NBUF; ++b) mbar_init(&full[b], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    __syncthreads();
    const int J = NPH * ((M + NGRP - 1) / NGRP), Q = J * NGRP;
    auto decode = [&](int q) { LpTask t; const int j = q / NGRP; t.m = q % NGRP + NGRP * (j / NPH); t.phase = j % NPH; t.valid = t.m < M; return t; };
    auto fill = [&](int q) {
        const LpTask t = decode(q);
        const int b = q % NBUF;
        if (t.valid) issue(t, smem + b * SM::BUF_BYTES, &full[b]); else mbar_arrive(&full[b]);
    };
    if (threadIdx.x == 0)
        for (int q = 0; q < NBUF && q < Q; ++q) fill(q);
    const int gr = threadIdx.x / Cfg::GROUP_THREADS;
    for (int j = 0; j < J; ++j) {
        const int q = j * NGRP + gr, b = q % NBUF;
        const LpTask t = decode(q);
        mbar_wait(&full[b], (q / NBUF) & 1);
        if (t.valid) work(t, smem + b * SM::BUF_BYTES);
        if (line_tid<Cfg>() == 0 && q + NBUF < Q) { fence_proxy_async(); fill(q + NBUF); }
    }
}

// B3 inverse row FFT + B4 (k_adj_rows, kernels_nufft.cu) on the pipeline.  Input: the adjoint half-plane rowbuf[g][x][i]; row i,
// phase p takes x = 2 k + p, k < n: one 4-D tensor box {8 floats, 1 row i, 1 parity, 256 k} per 256 elements.
template <class Cfg, int NGRP, int NBUF>
__global__ void __launch_bounds__(NGRP * Cfg::GROUP_THREADS, 1) k_adj_rows_tma(DevPlan d, const __grid_constant__ CUtensorMap tm, int S, int ng,
                                                                             float *vol) {
    extern __shared__ __align__(128) char lt_smem[];
    const PlaneMajorLast<Cfg> cfg{};
    constexpr int n = Cfg::n(), R0 = Cfg::radix(0);
    const int nlines = n * ng;
    if ((int)blockIdx.x >= nlines) return;
    const int M = (nlines - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;
    const int tid = line_tid<Cfg>(), pl = tid % Cfg::PL, plo = tid / Cfg::SLOTS;     // plane in the passes / in the plane-major last pass
    line_pipeline<Cfg, NGRP, NBUF, 2>(lt_smem, M,
        [&](const LpTask &t, char *buf, unsigned long long *bar) {
            const int line = blockIdx.x + t.m * gridDim.x, g = line / n, i = line - g * n;
            mbar_arrive_expect_tx(bar, n * 32);
#pragma unroll
            for (int k0 = 0; k0 < n; k0 += LT_BOX_ROWS) tma_load_4d(buf + k0 * 32, &tm, 0, i, t.phase, g * n + k0, bar);
        },
        [&](const LpTask &t, char *buf) {
            const int line = blockIdx.x + t.m * gridDim.x, g = line / n, i = line - g * n, p = t.phase;
            float2 *sm = reinterpret_cast<float2 *>(buf);
            const LineCtx c = line_ctx<PlaneMajorLast<Cfg>>(sm, d.twG);
            const float di = d.deapod[i];
            const int sre = 8 * g + 2 * plo;
            const bool hre = sre < S, him = sre + 1 < S;
            float *vre = vol + ((size_t)sre * n + i) * n, *vim = vre + (size_t)n * n;
            line_first_inplace<R0, true>(c, cfg, [&](int k, bool) { return sm[k * 4 + pl]; });
            static_finish<true, PlaneMajorLast<Cfg>, 1, R0>(c, cfg,
                [&](int tt, bool lo) {                                              // this thread wrote them in phase 0
                    const int j = wrapped(tt, n, lo).img;
                    return p ? make_float2(hre ? vre[j] : 0.f, him ? vim[j] : 0.f) : make_float2(0.f, 0.f);
                },
                [&](int tt, bool lo, float2 v, float2 old) {
                    const Wrapped w = wrapped(tt, n, lo);
                    const float sc = di * __ldg(&d.deapod[w.img]);
                    if (p) v = cmulc(v, __ldg(&d.twG[w.X]));
                    v.x = fmaf(v.x, sc, old.x); v.y = fmaf(v.y, sc, old.y);
                    if (hre) vre[w.img] = v.x;
                    if (him) vim[w.img] = v.y;
                });
            line_sync<PlaneMajorLast<Cfg>>();                                      // the last pass has read the buffer
        });
}

template <int N>
static bool launch_adj_rows_tma_n(const DevPlan &d, const float2 *rowbuf, int S, int ng, float *vol, cudaStream_t st) {
    tc_encode_tiled_fn enc = tensor_map_encoder();
    if (!enc) return false;
    using L = LtSize<N, 2>;
    static thread_local LtMapCache c;          // per host thread: plans may be used from different threads (one plan, one thread at a time)
    if (c.ptr != rowbuf || c.ng != ng) {
        const cuuint64_t n = d.n;
        const cuuint64_t dims[4] = {8, n, 2, n * ng};
        const cuuint64_t strides[3] = {32, n * 32, 2 * n * 32};
        const cuuint32_t box[4] = {8, 1, 1, LT_BOX_ROWS}, es[4] = {1, 1, 1, 1};
        if (enc(&c.tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, const_cast<float2 *>(rowbuf), dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS) { c.ptr = nullptr; return false; }
        c.ptr = rowbuf; c.ng = ng;
    }
    constexpr int sh = LpSmem<N, L::NBUF>::TOTAL;
    static bool attr = false;
    if (!attr) { cudaFuncSetAttribute(k_adj_rows_tma<typename L::Cfg, L::NGRP, L::NBUF>, cudaFuncAttributeMaxDynamicSharedMemorySize, sh); attr = true; }
    k_adj_rows_tma<typename L::Cfg, L::NGRP, L::NBUF><<<std::min(lt_sm_count(), d.n * ng), L::NGRP * L::Cfg::GROUP_THREADS, sh, st>>>(d, c.tm, S, ng, vol);
    TC_COUNT_LAUNCH();
    return true;
}
static bool launch_adj_rows_tma(const DevPlan &d, const float2 *rowbuf, int S, int ng, float *vol, cudaStream_t st) {
    switch (d.n) {
    case 2048: return launch_adj_rows_tma_n<2048>(d, rowbuf, S, ng, vol, st);
    case 1024: return launch_adj_rows_tma_n<1024>(d, rowbuf, S, ng, vol, st);
    default: return false;
    }
}

// B3 inverse column FFT (k_adj_cols) on the pipeline.  Input: column x of the fine grid, phase p = the contiguous run of cells
// y = 2 k + p at grid[g][x][p n + k]; only the cells inside the sampled disc are brought in (one or two plain bulk copies).
template <class Cfg, int NGRP, int NBUF>
__global__ void __launch_bounds__(NGRP * Cfg::GROUP_THREADS, 1) k_adj_cols_tma(DevPlan d, const float2 *__restrict__ grid, int ng, float2 *rowbuf) {
    extern __shared__ __align__(128) char lt_smem[];
    const Cfg cfg{};
    constexpr int n = Cfg::n(), G = 2 * n, R0 = Cfg::radix(0);
    const int nlines = G * ng;
    if ((int)blockIdx.x >= nlines) return;
    const int M = (nlines - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;
    const int pl = line_tid<Cfg>() % Cfg::PL;
    line_pipeline<Cfg, NGRP, NBUF, 2>(lt_smem, M,
        [&](const LpTask &t, char *buf, unsigned long long *bar) {
            const int line = blockIdx.x + t.m * gridDim.x, g = line / G, x = line - g * G, p = t.phase;
            const int lim = disc_limit(x, G, d.discR);
            // live cells: k <= k1 (ky = 2 k + p >= 0) and k >= k2 (ky = 2 k + p - G < 0); found with disc_live itself
            int K = (int)sqrtf((float)lim);
            while ((K + 1) * (K + 1) <= lim) ++K;
            while (K * K > lim) --K;
            int k1 = (min(K, G / 2 - 1) - p) >> 1;                      // largest k with 2 k + p <= min(K, G/2 - 1); -1 if none
            if (min(K, G / 2 - 1) - p < 0) k1 = -1;
            int k2 = (max(G - K, G / 2) - p + 1) >> 1;                  // smallest k with 2 k + p >= max(G - K, G/2)
            if (k2 <= k1 + 1) { k1 = n - 1; k2 = n; }                   // the two runs touch: one copy
            const char *src = reinterpret_cast<const char *>(grid + (((size_t)g * G + x) * G + (size_t)p * n) * 4);
            mbar_arrive_expect_tx(bar, (unsigned)((k1 + 1 + n - k2) * 32));
            if (k1 >= 0) bulk_g2s(buf, src, (unsigned)(k1 + 1) * 32, bar);
            if (k2 < n) bulk_g2s(buf + (size_t)k2 * 32, src + (size_t)k2 * 32, (unsigned)(n - k2) * 32, bar);
        },
        [&](const LpTask &t, char *buf) {
            const int line = blockIdx.x + t.m * gridDim.x, g = line / G, x = line - g * G, p = t.phase;
            float2 *sm = reinterpret_cast<float2 *>(buf);
            const LineCtx c = line_ctx<Cfg>(sm, d.twG);
            const int lim = disc_limit(x, G, d.discR);
            float2 *out = rowbuf + ((size_t)g * G + x) * n * 4 + pl;                 // adjoint half-plane, column-major: [g][x][i]
            line_first_inplace<R0, true>(c, cfg, [&](int k, bool) { return disc_live(2 * k + p, G, lim) ? sm[k * 4 + pl] : make_float2(0.f, 0.f); });
            static_finish<true, Cfg, 1, R0>(c, cfg,
                [&](int tt, bool lo) { return p ? out[wrapped(tt, n, lo).img * 4] : make_float2(0.f, 0.f); },   // this thread wrote it in phase 0
                [&](int tt, bool lo, float2 v, float2 old) {
                    const Wrapped w = wrapped(tt, n, lo);
                    if (p) { v = cmulc(v, __ldg(&d.twG[w.X])); v = cadd(v, old); }
                    out[w.img * 4] = v;
                });
            line_sync<Cfg>();
        });
}

// Raw layout of a line that arrives as 8 float rows (one per slice of the group): row s at float offset s (n + 4), so that the
// four planes of a quad read four different bank groups.
template <int N> __device__ __forceinline__ int lt_frow(int s) { return s * (N + 4); }

// bulk copies of the rows of slices 8 g .. 8 g + 7 (those below S) of a [slice][line][n] float array
template <int N>
__device__ __forceinline__ void lt_issue_float_rows(const float *base, size_t slice_stride, size_t line_off, int g, int S, char *buf,
                                                    unsigned long long *bar) {
    const int ns = min(8, S - 8 * g);
    mbar_arrive_expect_tx(bar, (unsigned)ns * N * 4);
    for (int s = 0; s < ns; ++s)
        bulk_g2s(buf + (size_t)lt_frow<N>(s) * 4, base + (size_t)(8 * g + s) * slice_stride + line_off, N * 4, bar);
}

// F1 + row FFT (k_fwd_rows) on the pipeline: whole 32-byte cells are stored (4-plane groups).
template <class Cfg, int NGRP, int NBUF>
__global__ void __launch_bounds__(NGRP * Cfg::GROUP_THREADS, 1) k_fwd_rows_tma(DevPlan d, const float *__restrict__ vol, int S, int ng,
                                                                             float2 *__restrict__ rowbuf) {
    extern __shared__ __align__(128) char lt_smem[];
    const Cfg cfg{};
    constexpr int n = Cfg::n(), G = 2 * n, R0 = Cfg::radix(0);
    const int nlines = n * ng;
    if ((int)blockIdx.x >= nlines) return;
    const int M = (nlines - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;
    const int pl = line_tid<Cfg>() % Cfg::PL;
    line_pipeline<Cfg, NGRP, NBUF, 2>(lt_smem, M,
        [&](const LpTask &t, char *buf, unsigned long long *bar) {
            const int line = blockIdx.x + t.m * gridDim.x, g = line / n, i = line - g * n;
            lt_issue_float_rows<n>(vol, (size_t)n * n, (size_t)i * n, g, S, buf, bar);
        },
        [&](const LpTask &t, char *buf) {
            const int line = blockIdx.x + t.m * gridDim.x, g = line / n, i = line - g * n, p = t.phase;
            float2 *sm = reinterpret_cast<float2 *>(buf);
            const float *rf = reinterpret_cast<const float *>(buf);
            const LineCtx c = line_ctx<Cfg>(sm, d.twG);
            const float di = d.deapod[i];
            const int sre = 8 * g + 2 * pl;
            const bool hre = sre < S, him = sre + 1 < S;
            const float *rre = rf + lt_frow<n>(2 * pl), *rim = rf + lt_frow<n>(2 * pl + 1);
            float2 *out = rowbuf + ((size_t)g * n + i) * G * 4 + pl;
            line_first_inplace<R0, false>(c, cfg, [&](int tt, bool lo) {
                const Wrapped w = wrapped(tt, n, lo);
                const float sc = di * __ldg(&d.deapod[w.img]);
                float2 v = make_float2(hre ? rre[w.img] * sc : 0.f, him ? rim[w.img] * sc : 0.f);
                if (p) v = cmul(v, __ldg(&d.twG[w.X]));
                return v;
            });
            static_finish<false, Cfg, 1, R0>(c, cfg, NoPre(), [&](int r, bool, float2 v, float2) { out[(size_t)(p * n + r) * 4] = v; });
            line_sync<Cfg>();
        });
}

// B1 radial FFT + conjugate phase (k_adj_radial) on the pipeline: one phase per line (a, g).
template <class Cfg, int NGRP, int NBUF>
__global__ void __launch_bounds__(NGRP * Cfg::GROUP_THREADS, 1) k_adj_radial_tma(DevPlan d, const float *__restrict__ sino, int S, int ng,
                                                                               float2 *__restrict__ cpol) {
    extern __shared__ __align__(128) char lt_smem[];
    const Cfg cfg{};
    constexpr int nd = Cfg::n(), R0 = Cfg::radix(0);
    const int nlines = d.na * ng;
    if ((int)blockIdx.x >= nlines) return;
    const int M = (nlines - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;
    const int pl = line_tid<Cfg>() % Cfg::PL;
    line_pipeline<Cfg, NGRP, NBUF, 1>(lt_smem, M,
        [&](const LpTask &t, char *buf, unsigned long long *bar) {
            const int line = blockIdx.x + t.m * gridDim.x, g = line / d.na, a = line - g * d.na;
            lt_issue_float_rows<nd>(sino, (size_t)d.na * nd, (size_t)a * nd, g, S, buf, bar);
        },
        [&](const LpTask &t, char *buf) {
            const int line = blockIdx.x + t.m * gridDim.x, g = line / d.na, a = line - g * d.na;
            float2 *sm = reinterpret_cast<float2 *>(buf);
            const float *rf = reinterpret_cast<const float *>(buf);
            const LineCtx c = line_ctx<Cfg>(sm, d.twD);
            const int sre = 8 * g + 2 * pl;
            const bool hre = sre < S, him = sre + 1 < S;
            const float *rre = rf + lt_frow<nd>(2 * pl), *rim = rf + lt_frow<nd>(2 * pl + 1);
            float2 *out = cpol + ((size_t)g * d.na + a) * nd * 4 + pl;
            line_first_inplace<R0, false>(c, cfg, [&](int u, bool) { return make_float2(hre ? rre[u] : 0.f, him ? rim[u] : 0.f); });
            static_finish<false, Cfg, 1, R0>(c, cfg, NoPre(), [&](int k, bool, float2 v, float2) { out[(size_t)k * 4] = cmul(v, __ldg(&d.ph_adj[k])); });
            line_sync<Cfg>();
        });
}

// F4 centre phase + inverse radial FFT (k_fwd_radial) on the pipeline; plane-major last pass (whole 128-byte lines of one slice).
template <class Cfg, int NGRP, int NBUF>
__global__ void __launch_bounds__(NGRP * Cfg::GROUP_THREADS, 1) k_fwd_radial_tma(DevPlan d, const float2 *__restrict__ cpol, int S, int ng,
                                                                               float *__restrict__ sino) {
    extern __shared__ __align__(128) char lt_smem[];
    const PlaneMajorLast<Cfg> cfg{};
    constexpr int nd = Cfg::n(), R0 = Cfg::radix(0);
    const int nlines = d.na * ng;
    if ((int)blockIdx.x >= nlines) return;
    const int M = (nlines - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;
    const int tid = line_tid<Cfg>(), pl = tid % Cfg::PL, plo = tid / Cfg::SLOTS;
    line_pipeline<Cfg, NGRP, NBUF, 1>(lt_smem, M,
        [&](const LpTask &t, char *buf, unsigned long long *bar) {
            const int line = blockIdx.x + t.m * gridDim.x;
            mbar_arrive_expect_tx(bar, nd * 32);
            bulk_g2s(buf, cpol + (size_t)line * nd * 4, nd * 32, bar);
        },
        [&](const LpTask &t, char *buf) {
            const int line = blockIdx.x + t.m * gridDim.x, g = line / d.na, a = line - g * d.na;
            float2 *sm = reinterpret_cast<float2 *>(buf);
            const LineCtx c = line_ctx<PlaneMajorLast<Cfg>>(sm, d.twD);
            const int sre = 8 * g + 2 * plo;
            const bool hre = sre < S, him = sre + 1 < S;
            float *ore = sino + ((size_t)sre * d.na + a) * nd, *oim = ore + (size_t)d.na * nd;
            line_first_inplace<R0, true>(c, cfg, [&](int k, bool) {
                return 2 * k == nd ? make_float2(0.f, 0.f) : cmul(sm[k * 4 + pl], __ldg(&d.ph_fwd[k]));     // the Nyquist cell of cpol is never written
            });
            static_finish<true, PlaneMajorLast<Cfg>, 1, R0>(c, cfg, NoPre(), [&](int u, bool, float2 v, float2) {
                if (hre) ore[u] = v.x;
                if (him) oim[u] = v.y;
            });
            line_sync<PlaneMajorLast<Cfg>>();
        });
}

static bool lt_aligned16(const void *q) { return (reinterpret_cast<size_t>(q) & 15) == 0; }

// launch of a pipeline kernel KERNEL<Cfg, NGRP, NBUF> for line length N (twiddle stride TWS), `lines` lines
#define TC_LP_LAUNCH(KERNEL, N, TWS, lines, ...)                                                                              \
    do {                                                                                                                      \
        using L = LtSize<N, TWS>;                                                                                             \
        constexpr int sh = LpSmem<N, L::NBUF>::TOTAL;                                                                         \
        static bool attr = false;                                                                                             \
        if (!attr) { cudaFuncSetAttribute(KERNEL<typename L::Cfg, L::NGRP, L::NBUF>, cudaFuncAttributeMaxDynamicSharedMemorySize, sh); attr = true; } \
        KERNEL<typename L::Cfg, L::NGRP, L::NBUF><<<std::min(lt_sm_count(), (lines)), L::NGRP * L::Cfg::GROUP_THREADS, sh, st>>>(__VA_ARGS__);        \
        TC_COUNT_LAUNCH();                                                                                                    \
    } while (0)

static bool launch_adj_cols_tma(const DevPlan &d, const float2 *grid, int ng, float2 *rowbuf, cudaStream_t st) {
    switch (d.n) {
    case 2048: TC_LP_LAUNCH(k_adj_cols_tma, 2048, 2, d.G * ng, d, grid, ng, rowbuf); return true;
    case 1024: TC_LP_LAUNCH(k_adj_cols_tma, 1024, 2, d.G * ng, d, grid, ng, rowbuf); return true;
    default: return false;
    }
}
static bool launch_fwd_rows_tma(const DevPlan &d, const float *vol, int S, int ng, float2 *rowbuf, cudaStream_t st) {
    if (!lt_aligned16(vol)) return false;
    switch (d.n) {
    case 2048: TC_LP_LAUNCH(k_fwd_rows_tma, 2048, 2, d.n * ng, d, vol, S, ng, rowbuf); return true;
    case 1024: TC_LP_LAUNCH(k_fwd_rows_tma, 1024, 2, d.n * ng, d, vol, S, ng, rowbuf); return true;
    default: return false;
    }
}
static bool launch_adj_radial_tma(const DevPlan &d, const float *sino, int S, int ng, float2 *cpol, cudaStream_t st) {
    if (!lt_aligned16(sino)) return false;
    switch (d.nd) {
    case 2048: TC_LP_LAUNCH(k_adj_radial_tma, 2048, 1, d.na * ng, d, sino, S, ng, cpol); return true;
    case 1024: TC_LP_LAUNCH(k_adj_radial_tma, 1024, 1, d.na * ng, d, sino, S, ng, cpol); return true;
    default: return false;
    }
}
static bool launch_fwd_radial_tma(const DevPlan &d, const float2 *cpol, int S, int ng, float *sino, cudaStream_t st) {
    switch (d.nd) {
    case 2048: TC_LP_LAUNCH(k_fwd_radial_tma, 2048, 1, d.na * ng, d, cpol, S, ng, sino); return true;
    case 1024: TC_LP_LAUNCH(k_fwd_radial_tma, 1024, 1, d.na * ng, d, cpol, S, ng, sino); return true;
    default: return false;
    }
}
