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
//   shared memory: raw [n cells] | work 0 | work 1 | mbarriers      (n = 2048: 64 KB + 2 x 68 KB)

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
__global__ void __launch_bounds__(2 * Cfg::GROUP_THREADS, 1) k_fwd_cols_tma(DevPlan d, const __grid_constant__ CUtensorMap tm, int ng,
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
        const int lim = disc_limit(x, G);
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

// true if the TMA-fed kernel took the launch
static bool launch_fwd_cols_tma(const DevPlan &d, const float2 *rowbuf, int ng, float2 *grid, cudaStream_t st) {
    if (d.n != 2048) return false;
    tc_encode_tiled_fn enc = tensor_map_encoder();
    if (!enc) return false;
    using Cfg = Grouped<SCfg<4, 2048, 2, 16, 16, 8>, 512>;
    static const float2 *c_ptr = nullptr; static int c_ng = 0; static CUtensorMap c_tm;
    if (c_ptr != rowbuf || c_ng != ng) {
        const cuuint64_t dims[3] = {8, (cuuint64_t)d.G, (cuuint64_t)d.n * ng};
        const cuuint64_t strides[2] = {32, (cuuint64_t)d.G * 32};
        const cuuint32_t box[3] = {8, 1, LT_BOX_ROWS}, es[3] = {1, 1, 1};
        const int l2 = lt_l2_promotion();
        const CUtensorMapL2promotion pr = l2 == 1 ? CU_TENSOR_MAP_L2_PROMOTION_L2_64B : l2 == 2 ? CU_TENSOR_MAP_L2_PROMOTION_L2_128B
                                        : l2 == 3 ? CU_TENSOR_MAP_L2_PROMOTION_L2_256B : CU_TENSOR_MAP_L2_PROMOTION_NONE;
        if (enc(&c_tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<float2 *>(rowbuf), dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                CU_TENSOR_MAP_SWIZZLE_NONE, pr, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS) { c_ptr = nullptr; return false; }
        c_ptr = rowbuf; c_ng = ng;
    }
    static int n_sm = 0;
    if (!n_sm) { int dev = 0; cudaGetDevice(&dev); cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev); if (n_sm <= 0) n_sm = 148; }
    constexpr int sh = LtSmem<2048>::TOTAL;
    static bool attr = false;
    if (!attr) { cudaFuncSetAttribute(k_fwd_cols_tma<Cfg>, cudaFuncAttributeMaxDynamicSharedMemorySize, sh); attr = true; }
    k_fwd_cols_tma<Cfg><<<std::min(n_sm, d.G * ng), 2 * Cfg::GROUP_THREADS, sh, st>>>(d, c_tm, ng, grid);
    TC_COUNT_LAUNCH();
    return true;
}
