// Included by kernels_nufft.cu inside namespace tc: the forward polar gather (F3, eq. (7) reversed) binned by
// fine-grid tile, and F4 (centre phase + inverse radial FFT, eq. (6) reversed P:L81) as its own launch.
//
// Why: evaluated ray by ray (k_fwd_gather) every one of a sample's 36 taps is its own scattered 32-byte request; the L1 data pipe
// serves one 128-byte line per cycle whatever the request size, so that form is bound at 36 L1 wavefronts per sample and group,
// with most of them going on to L2.  Here a CTA owns a GT_CX x GT_CY tile of fine-grid cells (72 KB), brings it into shared
// memory ONCE with bulk asynchronous copies (cp.async.bulk -> UBLKCP, completion on an mbarrier; the rows are contiguous runs of
// 32-byte cells because the fast axis is parity-split), and serves every polar sample whose 6 x 6 taps lie in the tile from
// there: 128 bytes per shared-memory wavefront instead of 32, each cell crosses L2 -> SM once (plus the halo) instead of ~20
// times.  Tiles are multi-buffered: the copies of the next (tile, group) loads run while the current one is being read.
// The geometry (which samples a tile owns, their local tap base and fractional offsets) is plan-time data, shared by all groups
// and calls.  The price is one HBM round trip of the polar coefficients (cpol: 2 x 32 B per sample and group, ~4 % of the
// fine grid's bytes at config 4) between this kernel and k_fwd_radial.

// ---- plan-time tables -------------------------------------------------------------------------------------------------------
struct GtGeom { int bx, by; float rx, ry; };
// first tap and offsets of sample (a, m), decided in float64 exactly as k_fwd_gather / the oracle decide them (readings G6, G19)
__device__ __forceinline__ GtGeom gt_geom(const DevPlan &d, int a, int m) {
    const double2 cs = d.cs[a];
    const double kx = __dmul_rn((double)m, cs.x), ky = __dmul_rn((double)m, cs.y);      // rounded products: the same kappa as the spread's lists (enum_cell_taps)
    const double bxd = ceil(kx - d.hw), byd = ceil(ky - d.hw);
    GtGeom g; g.bx = (int)bxd; g.by = (int)byd; g.rx = (float)(kx - bxd); g.ry = (float)(ky - byd);
    return g;
}

// key = (tile << 32) | (a * nd + (m mod nd)); the excluded Nyquist mode (reading G2) sorts last
__global__ void k_gt_keys(DevPlan d, unsigned long long *__restrict__ keys) {
    const size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x;
    if (i >= (size_t)d.na * d.nd) return;
    const int a = (int)(i / d.nd), mi = (int)(i - (size_t)a * d.nd), m = mi - d.nd / 2;
    if (m == -d.nd / 2) { keys[i] = ~0ull; return; }
    const GtGeom g = gt_geom(d, a, m);
    const int tx = (g.bx - gt_min(d.G, d.W)) / GT_BX, ty = (g.by - gt_min(d.G, d.W)) / GT_BY;
    keys[i] = ((unsigned long long)(ty * d.gt_ntx + tx) << 32) | (unsigned)(a * d.nd + (m < 0 ? m + d.nd : m));
}

__global__ void k_gt_fill(DevPlan d, const unsigned long long *__restrict__ keys, unsigned nvalid, int4 *__restrict__ samples,
                          unsigned *__restrict__ counts) {
    const unsigned i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nvalid) return;
    const unsigned long long key = keys[i];
    const int tile = (int)(key >> 32), idx = (int)(key & 0xffffffffu);
    const int a = idx / d.nd, k = idx - a * d.nd, m = k < d.nd / 2 ? k : k - d.nd;
    const GtGeom g = gt_geom(d, a, m);
    const int tx = tile % d.gt_ntx, ty = tile / d.gt_ntx;
    const int lx = g.bx - (gt_min(d.G, d.W) + tx * GT_BX), ly = g.by - (gt_min(d.G, d.W) + ty * GT_BY);   // in [0, GT_BX) x [0, GT_BY)
    samples[i] = make_int4(idx, (ly << 16) | lx, __float_as_int(g.rx), __float_as_int(g.ry));
    atomicAdd(&counts[tile], 1u);
}

// ---- mbarrier / bulk-copy primitives (PTX; sm_90+) --------------------------------------------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long *bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(unsigned long long *bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long *bar, unsigned parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// global -> shared, `bytes` a multiple of 16, both addresses 16-byte aligned; completes `bytes` on the mbarrier
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, unsigned bytes, unsigned long long *bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// ---- the gather ---------------------------------------------------------------------------------------------------------------
// The kernel's x is the fine grid's FAST (contiguous, parity-split) axis and y its slow axis (rows), as in k_fwd_gather.
// Shared tile: cell (yl, xl) at ((yl * 2 + (xl & 1)) * (GT_CX / 2) + (xl >> 1)) * 32 bytes: the global row layout, cut to the tile.
constexpr int GT_THREADS = 1024;
template <int W> struct GtT {
    static constexpr int CX = GtDim<W>::CX, CY = GtDim<W>::CY;
    static constexpr int RUNS = CY * 2;                      // (row, parity) runs of CX / 2 cells each
    static constexpr int RUN_BYTES = (CX / 2) * 32;
    static constexpr int TILE_BYTES = CX * CY * 32;
    static_assert(RUNS <= GT_THREADS, "one thread per run");
    static_assert(GT_NBUF * TILE_BYTES + 64 <= 227 * 1024, "tiles must fit in shared memory");
};

template <int W>
__device__ __forceinline__ void gt_issue_tile(const DevPlan &d, const float2 *__restrict__ grid, int tile, int g, char *buf,
                                              unsigned long long *bar) {
    // threads 0 .. RUNS-1: one run each (two copies when the run wraps around the end of the parity block)
    constexpr int GT_CX = GtT<W>::CX, GT_RUNS = GtT<W>::RUNS, GT_RUN_BYTES = GtT<W>::RUN_BYTES;
    const int r = threadIdx.x;
    if (r >= GT_RUNS) return;
    const int G = d.G, nh = G >> 1;
    const int tx = tile % d.gt_ntx, ty = tile / d.gt_ntx;
    const int yl = r >> 1, par = r & 1;
    int Y = gt_min(G, W) + ty * GT_BY + yl;                                    // centred row -> storage row (taps wrap modulo G, reading G7)
    Y %= G; if (Y < 0) Y += G;
    int X = gt_min(G, W) + tx * GT_BX + par;                                   // first cell of the run (centred; same parity as par)
    X %= G; if (X < 0) X += G;
    const int pos0 = X >> 1;
    const int len1 = min(GT_CX / 2, nh - pos0), len2 = GT_CX / 2 - len1;
    const char *row = reinterpret_cast<const char *>(grid) + (((size_t)g * G + Y) * G + (size_t)par * nh) * 32;
    char *dst = buf + (size_t)r * GT_RUN_BYTES;
    mbar_arrive_expect_tx(bar, GT_RUN_BYTES);
    bulk_g2s(dst, row + (size_t)pos0 * 32, len1 * 32, bar);
    if (len2 > 0) bulk_g2s(dst + len1 * 32, row, len2 * 32, bar);
}

// Work items.  Tiles are sorted by sample count (most first).  One item = one tile for a run of GC consecutive groups, so that
// the thread pair that owns a sample evaluates its window weights ONCE and reuses them for every group of the run (the geometry
// is the same for all groups); the tiles near the origin, where every ray passes, are cut into shorter runs so that no item is
// more than a few per cent of a CTA's share: tile ranks [0, nh): GC = 1, [nh, nm): GC = 4, the rest: GC = 16.
// Items are dealt to the CTAs round robin, heavy ones first; a CTA streams the (tile, group) loads of its items through
// GT_NBUF shared-memory buffers, GT_NBUF - 1 loads ahead of the one being read.
struct GtCursor {
    int w, j, tile, g0, gc;            // item, position in its run of groups, tile id, first group, groups in this item
    bool valid;
};
__device__ __forceinline__ void gt_decode(const DevPlan &d, int ng, GtCursor &c) {
    const int c4 = (ng + 3) >> 2, c16 = (ng + 15) >> 4;
    const int nA = d.gt_nh * ng, nB = (d.gt_nm - d.gt_nh) * c4, nC = (d.gt_nlive - d.gt_nm) * c16;
    c.j = 0;
    c.valid = c.w < nA + nB + nC;
    if (!c.valid) return;
    int rank, step;
    if (c.w < nA) { rank = c.w / ng; c.g0 = c.w - rank * ng; step = 1; }
    else if (c.w < nA + nB) { const int v = c.w - nA; rank = v / c4; c.g0 = (v - rank * c4) * 4; rank += d.gt_nh; step = 4; }
    else { const int v = c.w - nA - nB; rank = v / c16; c.g0 = (v - rank * c16) * 16; rank += d.gt_nm; step = 16; }
    c.gc = min(step, ng - c.g0);
    c.tile = d.gt_tiles[rank];
}
__device__ __forceinline__ void gt_advance(const DevPlan &d, int ng, GtCursor &c) {
    if (++c.j < c.gc) return;
    c.w += gridDim.x;
    gt_decode(d, ng, c);
}

template <int W> struct GtTaps { float wx[W], wy[W]; int base; };          // window weights and the float4 index of tap (0, 0) in the tile
template <int W>
__device__ __forceinline__ GtTaps<W> gt_taps(const DevPlan &d, const int4 e) {
    constexpr int KB_W = W, GT_CX = GtT<W>::CX;
    GtTaps<W> t;
    const int lx = e.y & 0xffff, ly = e.y >> 16;
    const float rx = __int_as_float(e.z), ry = __int_as_float(e.w);
#pragma unroll
    for (int k = 0; k < KB_W; ++k) { t.wx[k] = kb_eval(d, rx - (float)k); t.wy[k] = kb_eval(d, ry - (float)k); }
    // cell (yl, xl) sits at float4 index (yl * GT_CX + (xl & 1) * (GT_CX / 2) + (xl >> 1)) * 2: taps t and t + 2 along x are neighbours
    t.base = (ly * GT_CX + (lx & 1) * (GT_CX / 2) + (lx >> 1)) * 2;
    return t;
}
// sum over the W x W taps; `odd` = parity of the first tap's column (decides on which side of the parity split taps 1, 3, 5 lie)
template <int W>
__device__ __forceinline__ float4 gt_apply(const float4 *__restrict__ tb, const GtTaps<W> &t, bool odd) {
    constexpr int KB_W = W, GT_CX = GtT<W>::CX;
    // x taps 0, 2, 4 share the parity of lx and sit at +0, +1, +2 cells; taps 1, 3, 5 have the other parity: the other run, and one cell
    // further along when lx is odd
    const int o1 = odd ? (1 - GT_CX / 2) * 2 : (GT_CX / 2) * 2;
    const float4 *p0 = tb + t.base, *p1 = p0 + o1;
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
    for (int ty = 0; ty < KB_W; ++ty) {
#pragma unroll
        for (int tx = 0; tx < KB_W; ++tx) {
            const float4 v = (tx & 1) ? p1[ty * GT_CX * 2 + (tx >> 1) * 2] : p0[ty * GT_CX * 2 + (tx >> 1) * 2];
            const float w2 = t.wy[ty] * t.wx[tx];
            acc.x = fmaf(w2, v.x, acc.x); acc.y = fmaf(w2, v.y, acc.y);
            acc.z = fmaf(w2, v.z, acc.z); acc.w = fmaf(w2, v.w, acc.w);
        }
    }
    return acc;
}

template <int W>
__global__ void __launch_bounds__(GT_THREADS, 1) k_fwd_gather_tiles(DevPlan d, const float2 *__restrict__ grid, int ng, float2 *__restrict__ cpol) {
    constexpr int GT_RUNS = GtT<W>::RUNS, GT_TILE_BYTES = GtT<W>::TILE_BYTES;
    extern __shared__ __align__(128) char gt_smem[];
    char *tiles = gt_smem;                                                 // GT_NBUF x GT_TILE_BYTES
    unsigned long long *bars = reinterpret_cast<unsigned long long *>(gt_smem + GT_NBUF * GT_TILE_BYTES);
    if (threadIdx.x == 0)
        for (int b = 0; b < GT_NBUF; ++b) mbar_init(&bars[b], GT_RUNS);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    __syncthreads();
    const int pair = threadIdx.x >> 1, hp = threadIdx.x & 1;
    const size_t gstride = (size_t)d.na * d.nd * 2;                        // float4 units per group of cpol
    GtCursor cons, prod;
    cons.w = blockIdx.x; gt_decode(d, ng, cons);
    prod = cons;
    // prologue: GT_NBUF - 1 loads are on their way before the first one is read
#pragma unroll
    for (int j = 0; j < GT_NBUF - 1; ++j)
        if (prod.valid) { gt_issue_tile<W>(d, grid, prod.tile, prod.g0 + prod.j, tiles + j * GT_TILE_BYTES, &bars[j]); gt_advance(d, ng, prod); }
    GtTaps<W> mine;                                                           // this pair's first sample of the current tile, kept across its groups
    int mine_idx = -1; bool mine_odd = false;
    unsigned s0 = 0, s1 = 0;
    for (int k = 0; cons.valid; ++k) {
        if (prod.valid) {                                                  // that buffer was released by the barrier that ended load k - 1
            fence_proxy_async();
            const int bn = (k + GT_NBUF - 1) % GT_NBUF;
            gt_issue_tile<W>(d, grid, prod.tile, prod.g0 + prod.j, tiles + bn * GT_TILE_BYTES, &bars[bn]);
            gt_advance(d, ng, prod);
        }
        if (cons.j == 0) {                                                 // new tile: weights of this pair's first sample
            s0 = d.gt_start[cons.tile]; s1 = d.gt_start[cons.tile + 1];
            mine_idx = -1;
            if (s0 + pair < s1) {
                const int4 e = __ldg(&d.gt_samples[s0 + pair]);
                mine = gt_taps<W>(d, e); mine_idx = e.x; mine_odd = e.y & 1;
            }
        }
        const int bc = k % GT_NBUF;
        const float4 *tb = reinterpret_cast<const float4 *>(tiles + bc * GT_TILE_BYTES) + hp;
        float4 *out = reinterpret_cast<float4 *>(cpol) + (size_t)(cons.g0 + cons.j) * gstride + hp;
        mbar_wait(&bars[bc], (k / GT_NBUF) & 1);
        if (mine_idx >= 0) out[(size_t)mine_idx * 2] = gt_apply<W>(tb, mine, mine_odd);
#pragma unroll 1
        for (unsigned s = s0 + pair + GT_THREADS / 2; s < s1; s += GT_THREADS / 2) {       // crowded tiles: the further samples of this pair
            const int4 e = __ldg(&d.gt_samples[s]);
            const GtTaps<W> t = gt_taps<W>(d, e);
            out[(size_t)e.x * 2] = gt_apply<W>(tb, t, e.y & 1);
        }
        __syncthreads();                                                   // everybody is done reading this buffer
        gt_advance(d, ng, cons);
    }
}

// F4: p[a][u] = (1/nd) sum_m c[a][m] e^{2 pi i m (u - centre)/nd}  (phase table ph_fwd carries 1/nd and the centre shift; its Nyquist
// entry is 0 and that cell of cpol is never written, so it is not read either).  grid = (na, ng).
template <class Cfg>
__global__ void TC_LB k_fwd_radial(DevPlan d, const float2 *__restrict__ cpol, int S, float *__restrict__ sino) {
    float2 *sm = reinterpret_cast<float2 *>(smem_f4);
    const Cfg cfg = make_cfg<Cfg>(d.fD, 1);
    const int a = blockIdx.x, g = blockIdx.y, nd = cfg.n(), pl = threadIdx.x & 3;
    const int sre = 8 * g + 2 * pl;
    const bool hre = sre < S, him = sre + 1 < S;
    const float2 *in = cpol + ((size_t)g * d.na + a) * nd * 4 + pl;
    float *ore = sino + ((size_t)sre * d.na + a) * nd, *oim = ore + (size_t)d.na * nd;
    fft_line<true>(sm, cfg, d.twD,
        [&](int k, bool) { return 2 * k == nd ? make_float2(0.f, 0.f) : cmul(__ldg(&in[(size_t)k * 4]), __ldg(&d.ph_fwd[k])); },
        NoPre(), [&](int u, bool, float2 v, float2) {
            if (hre) ore[u] = v.x;
            if (him) oim[u] = v.y;
        });
}

static bool launch_fwd_radial_tma(const DevPlan &d, const float2 *cpol, int S, int ng, float *sino, cudaStream_t st);   // kernels_line_tma.cuh
void launch_fwd_radial(const DevPlan &d, const float2 *cpol, int S, int ng, float *sino, cudaStream_t st) {
    static const bool plain = env_is("TC_FRAD", "plain");
    if (!plain && launch_fwd_radial_tma(d, cpol, S, ng, sino, st)) return;
    TC_LINE_LAUNCH(k_fwd_radial, 4, 1, 0, d.fD, dim3(d.na, ng), d, cpol, S, sino);
}
void launch_gt_keys(const DevPlan &d, unsigned long long *keys, cudaStream_t st) {
    const size_t n = (size_t)d.na * d.nd;
    k_gt_keys<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(d, keys);
}
void launch_gt_fill(const DevPlan &d, const unsigned long long *keys, unsigned nvalid, int4 *samples, unsigned *counts, cudaStream_t st) {
    k_gt_fill<<<(nvalid + 255) / 256, 256, 0, st>>>(d, keys, nvalid, samples, counts);
}
template <int W>
static void launch_fwd_gather_tiles_w(const DevPlan &d, const float2 *grid, int ng, float2 *cpol, int nitems, int n_sm, cudaStream_t st) {
    const size_t sh = GT_NBUF * GtT<W>::TILE_BYTES + 64;
    static bool attr = false;
    if (!attr) { cudaFuncSetAttribute(k_fwd_gather_tiles<W>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sh); attr = true; }
    k_fwd_gather_tiles<W><<<std::min(n_sm, nitems), GT_THREADS, sh, st>>>(d, grid, ng, cpol);
}
void launch_fwd_gather_tiles(const DevPlan &d, const float2 *grid, int ng, float2 *cpol, cudaStream_t st) {
    static int n_sm = 0;
    if (!n_sm) { int dev = 0; cudaGetDevice(&dev); cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev); if (n_sm <= 0) n_sm = 148; }
    const int nitems = d.gt_nh * ng + (d.gt_nm - d.gt_nh) * ((ng + 3) / 4) + (d.gt_nlive - d.gt_nm) * ((ng + 15) / 16);
    if (nitems <= 0) return;
    if (d.W == 4) launch_fwd_gather_tiles_w<4>(d, grid, ng, cpol, nitems, n_sm, st);
    else if (d.W == 8) launch_fwd_gather_tiles_w<8>(d, grid, ng, cpol, nitems, n_sm, st);
    else launch_fwd_gather_tiles_w<6>(d, grid, ng, cpol, nitems, n_sm, st);
    TC_COUNT_LAUNCH();
}
