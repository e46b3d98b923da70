// Included by kernels_nufft.cu inside namespace tc: polar-side kernels (F3+F4, B1, B2) and launch wrappers.

// Kaiser-Bessel window phi(r), |r| <= W/2 (reading G5): degree-12 polynomial in z = 2 q - 1,
// q = 1 - (2 r / W)^2, fitted in float64 at plan creation (max error 3e-10 before float32 rounding).
__device__ __forceinline__ float kb_eval(const DevPlan &d, float r) {      // coefficients ride in the plan (kernel parameter space)
    const float z = fmaf(r * r, d.kbs, 1.f);
    float acc = d.kb[KB_DEG];
#pragma unroll
    for (int k = KB_DEG - 1; k >= 0; --k) acc = fmaf(acc, z, d.kb[k]);
    return acc;
}

// ------------------------------------------------------------------------------------------------
// The polar kernels see the fine grid transposed (grid[g][x][y...]: slow index = x, fast index = y), so the plan
// hands them the rays of theta' = pi/2 - theta: their "kx" below is the true k_y and vice versa.
// F3 polar gather (eq. (7) reversed) fused with F4 centre phase + inverse radial FFT
// (eq. (6) reversed P:L81, shift property).  grid = (na, ng); the radial line of all P planes
// stays in shared memory, so polar coefficients never reach HBM on the forward side.
// One CTA of 1024 threads per SM rather than two of 512: the same warps, but half the shared memory, and the gather lives on
// L1 (measured: 9.9 ms with no L1, 4.34 ms with two CTAs, 4.13 ms with one).  The radial FFT uses the first SLOTS * 4 threads.
constexpr int GATHER_THREADS = 1024;
template <class Cfg>
__global__ void __launch_bounds__(GATHER_THREADS, 1) k_fwd_gather(DevPlan d, const float2 *__restrict__ grid, int S, float *__restrict__ sino) {
    float2 *sm = reinterpret_cast<float2 *>(smem_f4);
    const int a = blockIdx.x, g = blockIdx.y;
    const Cfg cfg = make_cfg<Cfg>(d.fD, 1);
    const int nd = cfg.n(), G = d.G, R1 = cfg.radix(0);
    const double2 cs = d.cs[a];
    const float4 *gg = reinterpret_cast<const float4 *>(grid) + (size_t)g * G * G * 2;
    const int nh = G >> 1;                                     // fast axis is parity-split: index i sits at (i & 1) nh + (i >> 1)
    // two lanes per polar sample: lane parity = which 16-byte half of every 32-byte cell (planes 2hp, 2hp+1),
    // so one load instruction touches one sector per sample and needs no cross-lane reduction
    const int hp = threadIdx.x & 1;
    for (int mi = threadIdx.x >> 1; mi < nd; mi += blockDim.x >> 1) {
        const int m = mi - nd / 2;
        const int k = m < 0 ? m + nd : m;
        float4 *dst = reinterpret_cast<float4 *>(sm + (size_t)line_input_cell(nd, R1, k) * 4) + hp;
        if (m == -nd / 2) { *dst = make_float4(0.f, 0.f, 0.f, 0.f); continue; }     // Nyquist radial mode excluded (reading G2)
        const double kx = __dmul_rn((double)m, cs.x), ky = __dmul_rn((double)m, cs.y);   // kappa = G k_m (cos, sin), in fine-grid cells (rounded product, see enum_cell_taps)
        const double bxd = ceil(kx - 3.0), byd = ceil(ky - 3.0);   // first tap (reading G6)
        const float rx = (float)(kx - bxd), ry = (float)(ky - byd);   // in (2, 3]
        const int bx = (int)bxd, by = (int)byd;
        float wx[KB_W], wy[KB_W];
#pragma unroll
        for (int t = 0; t < KB_W; ++t) { wx[t] = kb_eval(d, rx - (float)t); wy[t] = kb_eval(d, ry - (float)t); }
        float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
        int ixs[KB_W];
#pragma unroll
        for (int t = 0; t < KB_W; ++t) { const int ix = wrap(bx + t, G); ixs[t] = ((ix & 1) * nh + (ix >> 1)) * 2 + hp; }
#pragma unroll
        for (int ty = 0; ty < KB_W; ++ty) {
            const int iy = wrap(by + ty, G);
            const float4 *row = gg + (size_t)iy * G * 2;
#pragma unroll
            for (int tx = 0; tx < KB_W; ++tx) {
                const float4 v = __ldg(row + ixs[tx]);
                const float w = wy[ty] * wx[tx];
                acc.x = fmaf(w, v.x, acc.x); acc.y = fmaf(w, v.y, acc.y);
                acc.z = fmaf(w, v.z, acc.z); acc.w = fmaf(w, v.w, acc.w);
            }
        }
        const float2 ph = __ldg(&d.ph_fwd[k]);
        const float2 c0 = cmul(make_float2(acc.x, acc.y), ph), c1 = cmul(make_float2(acc.z, acc.w), ph);
        *dst = make_float4(c0.x, c0.y, c1.x, c1.y);
    }
    __syncthreads();
    {
        const int pl = threadIdx.x & 3, sre = 8 * g + 2 * pl;
        const bool hre = sre < S, him = sre + 1 < S;
        float *ore = sino + ((size_t)sre * d.na + a) * nd, *oim = ore + (size_t)d.na * nd;
        fft_line_from_smem<true>(sm, cfg, d.twD, [&](int u, bool, float2 v, float2) {
            if (hre) ore[u] = v.x;
            if (him) oim[u] = v.y;
        });
    }
}

// B1 radial FFT + conjugate phase (eq. (6)): c[a][m] = (1/nd) sum_u y[a][u] e^{-2 pi i m (u - centre)/nd}.
// grid = (na, ng).  cpol[((g na + a) nd + (m mod nd)) P + p].
template <class Cfg>
__global__ void TC_LB k_adj_radial(DevPlan d, const float *__restrict__ sino, int S, float2 *__restrict__ cpol) {
    float2 *sm = reinterpret_cast<float2 *>(smem_f4);
    const Cfg cfg = make_cfg<Cfg>(d.fD, 1);
    const int a = blockIdx.x, g = blockIdx.y, nd = cfg.n(), pl = threadIdx.x & 3;
    const int sre = 8 * g + 2 * pl;
    const bool hre = sre < S, him = sre + 1 < S;
    const float *ire = sino + ((size_t)sre * d.na + a) * nd, *iim = ire + (size_t)d.na * nd;
    float2 *out = cpol + ((size_t)g * d.na + a) * nd * 4 + pl;
    fft_line<false>(sm, cfg, d.twD,
        [&](int u, bool) { return make_float2(hre ? __ldg(&ire[u]) : 0.f, him ? __ldg(&iim[u]) : 0.f); },
        NoPre(), [&](int k, bool, float2 v, float2) { out[(size_t)k * 4] = cmul(v, __ldg(&d.ph_adj[k])); });
}

// ------------------------------------------------------------------------------------------------
// B2 polar -> Cartesian spread (eq. (7)), evaluated per fine-grid cell.  The type-1 sum
// Ghat[r] = sum_{(a,m): kappa - r in (-3,3]^2} c[a][m] phi phi is gathered by the thread that owns cell r:
// a tile of 32 x 8 cells bins the angles whose ray crosses the tile (one contiguous range of the
// angle list sorted by theta mod pi), each cell rejects rays that miss its own 6 x 6 box with one
// cross product, then solves for the <= 5 radial modes m on the dominant axis.  Accumulation is in
// registers, each cell is written once with a plain 32-byte store: no atomics, deterministic.
__device__ void tile_range(const DevPlan &d, double xa, double xb, double ya, double yb, int &start, int &count) {
    const double PI = 3.14159265358979323846;
    const int na = d.na;
    if (xa <= 0 && xb >= 0 && ya <= 0 && yb >= 0) { start = 0; count = na; return; }
    const double cx = 0.5 * (xa + xb), cy = 0.5 * (ya + yb);
    const double phic = atan2(cy, cx);
    double dmin = 1e30, dmax = -1e30;
    const double X[2] = {xa, xb}, Y[2] = {ya, yb};
    for (int i = 0; i < 2; ++i)
        for (int j = 0; j < 2; ++j) {
            const double dl = atan2(cx * Y[j] - cy * X[i], cx * X[i] + cy * Y[j]);
            dmin = fmin(dmin, dl); dmax = fmax(dmax, dl);
        }
    double lo = phic + dmin - 1e-4;
    const double w = dmax - dmin + 2e-4;
    if (w >= PI) { start = 0; count = na; return; }
    lo -= floor(lo / PI) * PI;
    const float lof = (float)lo;
    int l = 0, r = na;                                       // lower_bound(th_sorted, lo)
    while (l < r) { int mid = (l + r) >> 1; if (d.th_sorted[mid] < lof) l = mid + 1; else r = mid; }
    start = l;
    double hi = lo + w;
    const bool wrapd = hi >= PI;
    const float hif = (float)(wrapd ? hi - PI : hi);
    l = 0; r = na;                                           // upper_bound(th_sorted, hi)
    while (l < r) { int mid = (l + r) >> 1; if (d.th_sorted[mid] <= hif) l = mid + 1; else r = mid; }
    count = wrapd ? (na - start) + l : l - start;
    count = max(0, min(count, na));
}

// Tile ranges depend on the geometry only: computed once per plan (one thread per 32 x 8 tile).
__global__ void k_tile_ranges(DevPlan d, TileRange *__restrict__ rng, int *__restrict__ nrng) {
    const int G = d.G, tx = blockIdx.x * blockDim.x + threadIdx.x, ntx = (G + 31) / 32, nty = (G + 7) / 8;
    if (tx >= ntx * nty) return;
    const int bx = (tx % ntx) * 32, by = (tx / ntx) * 8;
    const int X0 = bx < G / 2 ? bx : bx - G, Y0 = by < G / 2 ? by : by - G;
    const int X1 = min(X0 + 31, G / 2 - 1), Y1 = min(Y0 + 7, G / 2 - 1);
    int shx[3] = {0, 0, 0}, shy[3] = {0, 0, 0}, nx = 1, ny = 1;
    const int hwi = d.W / 2;
    if (X0 <= -G / 2 + hwi) shx[nx++] = G;               // taps wrap modulo G (reading G7)
    if (X1 >= G / 2 - hwi - 1) shx[nx++] = -G;
    if (Y0 <= -G / 2 + hwi) shy[ny++] = G;
    if (Y1 >= G / 2 - hwi - 1) shy[ny++] = -G;
    int nr = 0;
    for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) {
            TileRange t; t.shx = shx[i]; t.shy = shy[j];
            tile_range(d, X0 + shx[i] - d.hw, X1 + shx[i] + d.hw, Y0 + shy[j] - d.hw, Y1 + shy[j] + d.hw, t.start, t.count);
            if (t.count > 0 && nr < 4) rng[tx * 4 + nr++] = t;
        }
    nrng[tx] = nr;
}

// Enumerates, for the cell owned by this thread, every polar sample (a, m) whose W x W footprint covers it
// (kappa - r in (-W/2, W/2]^2, decided in float64 exactly as the forward gather decides its tap base), and calls
// f(a * nd + (m mod nd), phi(dx) phi(dy)).  Cell order inside a tile: warp = 8 x 4 cells.
template <class F>
__device__ __forceinline__ void enum_cell_taps(const DevPlan &d, const TileRange *__restrict__ rng, const int *__restrict__ nrng,
                                               int tile, int ix, int iy, F f) {
    const int G = d.G, nd = d.nd, na = d.na;
    const int Kx0 = ix < G / 2 ? ix : ix - G, Ky0 = iy < G / 2 ? iy : iy - G;
    const int mmax = nd / 2 - 1, J = d.J;
    const int nr = nrng[tile];
    for (int e = 0; e < nr; ++e) {
        const TileRange tr = rng[tile * 4 + e];
        const int Kx = Kx0 + tr.shx, Ky = Ky0 + tr.shy;
        const float Kxf = (float)Kx, Kyf = (float)Ky;
        for (int i = 0; i < tr.count; ++i) {
            int k = tr.start + i; if (k >= na) k -= na;
            const double2 cs = d.cs_sorted[k];
            const float cf = (float)cs.x, sf = (float)cs.y;
            const float acf = fabsf(cf), asf = fabsf(sf);
            if (fabsf(Kxf * sf - Kyf * cf) > d.hwf * (acf + asf) + 0.02f) continue;   // ray misses this cell's box
            const float mc = acf >= asf ? Kxf / cf : Kyf / sf;
            const int m_c = __float2int_rn(mc);
            const int a = d.a_sorted[k];
            for (int j = -J - 1; j <= J + 1; ++j) {
                const int m = m_c + j;
                if (m < -mmax || m > mmax) continue;
                // kappa as the ROUNDED product (no fused multiply-add): the count and fill passes and the forward gather must take the
                // same decision for a sample that sits exactly on the edge of the window
                const double dx = __dmul_rn((double)m, cs.x) - Kx, dy = __dmul_rn((double)m, cs.y) - Ky;
                if (dx <= -d.hw || dx > d.hw || dy <= -d.hw || dy > d.hw) continue;
                f(a * nd + (m < 0 ? m + nd : m), kb_eval(d, (float)dx) * kb_eval(d, (float)dy));
            }
        }
    }
}

__device__ __forceinline__ void spread_cell(int &ix, int &iy, int &tile, int &cidx) {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    ix = blockIdx.x * 32 + (warp & 3) * 8 + (lane & 7);
    iy = blockIdx.y * 8 + (warp >> 2) * 4 + (lane >> 3);
    tile = blockIdx.y * gridDim.x + blockIdx.x;
    cidx = tile * 256 + threadIdx.x;
}

// Plan-time passes: count the taps of every cell, then (after an exclusive scan) write the (sample, weight) lists.
__global__ void __launch_bounds__(256) k_spread_count(DevPlan d, const TileRange *__restrict__ rng, const int *__restrict__ nrng, int *__restrict__ counts) {
    int ix, iy, tile, cidx; spread_cell(ix, iy, tile, cidx);
    int n = 0;
    if (ix < d.G && iy < d.G) enum_cell_taps(d, rng, nrng, tile, ix, iy, [&](int, float) { ++n; });
    counts[cidx] = n;
}
__global__ void __launch_bounds__(256) k_spread_fill(DevPlan d, const TileRange *__restrict__ rng, const int *__restrict__ nrng,
                                                     const unsigned *__restrict__ offs, int2 *__restrict__ taps) {
    int ix, iy, tile, cidx; spread_cell(ix, iy, tile, cidx);
    if (ix >= d.G || iy >= d.G) return;
    int2 *o = taps + offs[cidx];
    enum_cell_taps(d, rng, nrng, tile, ix, iy, [&](int idx, float w) { *o++ = make_int2(idx, __float_as_int(w)); });
}

// The hot kernel: a lane pair = one cell (lane parity = which 16-byte half of the cell).  A thread walks its cell's
// tap list (geometry-only, built once per plan, shared by every slice and every MBIR iteration) for GPT groups of
// 8 slices at a time, accumulates in registers and writes each cell with one plain 32-byte store per group.
// The kernel is bound by the chain of dependent loads (list offsets -> tap entries -> coefficients), so one
// thread serves ALL groups of the slab: the first 8 tap entries stay in registers across the group loop (a typical
// cell has 4-5 taps), longer lists are re-read from L2.  blockDim = 512.
template <int GPT>
__device__ __forceinline__ void spread_taps4(const int2 (&e)[4], const float4 *__restrict__ cg, const size_t (&qoff)[GPT], float4 (&acc)[GPT]) {
#pragma unroll
    for (int u = 0; u < 4; ++u) {
        const float4 *ca = cg + (size_t)e[u].x * 2;
        const float w = __int_as_float(e[u].y);
#pragma unroll
        for (int q = 0; q < GPT; ++q) {
            const float4 v = __ldg(ca + qoff[q]);
            acc[q].x = fmaf(w, v.x, acc[q].x); acc[q].y = fmaf(w, v.y, acc[q].y);
            acc[q].z = fmaf(w, v.z, acc[q].z); acc[q].w = fmaf(w, v.w, acc[q].w);
        }
    }
}

template <int GPT>
__global__ void __launch_bounds__(512, 2) k_adj_spread(DevPlan d, const unsigned *__restrict__ offs, const int2 *__restrict__ taps,
                                                       const float2 *__restrict__ cpol, int ng, float2 *__restrict__ grid) {
    const int c = threadIdx.x >> 1, hp = threadIdx.x & 1;
    const int warp = c >> 5, lane = c & 31;
    const int ix = blockIdx.x * 32 + (warp & 3) * 8 + (lane & 7), iy = blockIdx.y * 8 + (warp >> 2) * 4 + (lane >> 3);
    const int cidx = (blockIdx.y * gridDim.x + blockIdx.x) * 256 + c;
    const int G = d.G;
    if (ix >= G || iy >= G) return;
    const size_t gstride = (size_t)d.na * d.nd * 2;
    const unsigned t0 = offs[cidx], t1 = offs[cidx + 1];
    if (t1 - t0 > SPREAD_HEAVY) return;                          // long lists (cells near the origin) go to k_adj_spread_heavy
    if (t1 == t0) {                                              // outside the sampled disc: nobody reads the cell (see disc_live)
        const int kf = ix < G / 2 ? ix : ix - G, ks = iy < G / 2 ? iy : iy - G, R = d.discR;
        if (kf * kf + ks * ks > R * R) return;
    }
    // entries past the end of the list are (sample 0, weight 0)
    int2 e0[4], e1[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
        e0[u] = t0 + u < t1 ? __ldg(&taps[t0 + u]) : make_int2(0, 0);
        e1[u] = t0 + 4 + u < t1 ? __ldg(&taps[t0 + 4 + u]) : make_int2(0, 0);
    }
    float4 *out = reinterpret_cast<float4 *>(grid) + (((size_t)iy) * G + (ix & 1) * (G >> 1) + (ix >> 1)) * 2 + hp;
#pragma unroll 1
    for (int g0 = blockIdx.z * GPT; g0 < ng; g0 += GPT * gridDim.z) {
        float4 acc[GPT];
        size_t qoff[GPT];                                       // groups past the end re-read group g0 and are dropped at the store
#pragma unroll
        for (int q = 0; q < GPT; ++q) { acc[q] = make_float4(0.f, 0.f, 0.f, 0.f); qoff[q] = g0 + q < ng ? q * gstride : 0; }
        const float4 *cg = reinterpret_cast<const float4 *>(cpol) + (size_t)g0 * gstride + hp;
        if (t1 > t0) spread_taps4<GPT>(e0, cg, qoff, acc);
        if (t1 > t0 + 4) spread_taps4<GPT>(e1, cg, qoff, acc);
        for (unsigned t = t0 + 8; t < t1; t += 4) {
            int2 e[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) e[u] = t + u < t1 ? __ldg(&taps[t + u]) : make_int2(0, 0);
            spread_taps4<GPT>(e, cg, qoff, acc);
        }
#pragma unroll
        for (int q = 0; q < GPT; ++q)
            if (g0 + q < ng) out[(size_t)(g0 + q) * G * G * 2] = acc[q];
    }
}

// Cells whose list is longer than SPREAD_HEAVY taps (within ~90 cells of the origin, where every ray passes: 5 % of
// the taps, 0.2 % of the cells): one warp per cell and group block, fixed-order
// shuffle reduction, so the result stays deterministic and no thread of the main kernel runs a long serial loop.
__global__ void k_spread_heavy_list(DevPlan d, const unsigned *__restrict__ offs, unsigned ncell, unsigned *__restrict__ list, unsigned *__restrict__ count) {
    const unsigned c = blockIdx.x * blockDim.x + threadIdx.x;
    // a cell is listed if its own list or that of a cell of the same run (k_adj_spread_runs) is long
    if (c >= ncell) return;
    const unsigned c0 = c & ~(unsigned)(SP_NC - 1);
    bool heavy = false;
    for (unsigned k = c0; k < c0 + SP_NC; ++k) heavy = heavy || offs[k + 1] - offs[k] > SPREAD_HEAVY;
    if (heavy) list[atomicAdd(count, 1u)] = c;
}

template <int GPT>
__global__ void __launch_bounds__(256) k_adj_spread_heavy(DevPlan d, const unsigned *__restrict__ offs, const int2 *__restrict__ taps,
                                                          const unsigned *__restrict__ list, unsigned nheavy,
                                                          const float2 *__restrict__ cpol, int ng, float2 *__restrict__ grid) {
    // one warp per heavy cell and group block: 16 lane pairs stride through the list four entries at a time (the longest
    // lists, at the origin, have ~ 3 na taps), then a fixed-order shuffle reduction
    const unsigned wi = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (wi >= nheavy) return;
    const int lane = threadIdx.x & 31, hp = lane & 1, slot = lane >> 1;
    const unsigned cidx = list[wi];
    const int G = d.G, ntx = (G + 31) / 32;
    const int tile = cidx >> 8, c = cidx & 255, w = c >> 5, l = c & 31;
    const int ix = (tile % ntx) * 32 + (w & 3) * 8 + (l & 7), iy = (tile / ntx) * 8 + (w >> 2) * 4 + (l >> 3);
    const int g0 = blockIdx.y * GPT;
    const size_t gstride = (size_t)d.na * d.nd * 2;
    const float4 *cg = reinterpret_cast<const float4 *>(cpol) + (size_t)g0 * gstride + hp;
    float4 acc[GPT];
    size_t qoff[GPT];
#pragma unroll
    for (int q = 0; q < GPT; ++q) { acc[q] = make_float4(0.f, 0.f, 0.f, 0.f); qoff[q] = g0 + q < ng ? q * gstride : 0; }
    const unsigned t0 = offs[cidx], t1 = offs[cidx + 1];
    for (unsigned t = t0 + slot; t < t1; t += 64) {
        int2 e[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) e[u] = t + 16 * u < t1 ? __ldg(&taps[t + 16 * u]) : make_int2(0, 0);
        spread_taps4<GPT>(e, cg, qoff, acc);
    }
#pragma unroll
    for (int q = 0; q < GPT; ++q) {
#pragma unroll
        for (int o = 2; o < 32; o <<= 1) {
            acc[q].x += __shfl_xor_sync(0xffffffffu, acc[q].x, o); acc[q].y += __shfl_xor_sync(0xffffffffu, acc[q].y, o);
            acc[q].z += __shfl_xor_sync(0xffffffffu, acc[q].z, o); acc[q].w += __shfl_xor_sync(0xffffffffu, acc[q].w, o);
        }
        if (slot == 0 && g0 + q < ng)
            reinterpret_cast<float4 *>(grid)[(((size_t)(g0 + q) * G + iy) * G + (ix & 1) * (G >> 1) + (ix >> 1)) * 2 + hp] = acc[q];
    }
}

// ---- B2 by runs of cells (default) -----------------------------------------------------------------------------------------------
// k_adj_spread is bound by the L1 data pipe at one 32-byte sector per tap and group.  SP_NC cells next to each other along the fast
// axis share most of their samples (two cells: 42 instead of 72 per full footprint; four: 54 instead of 144), so a lane pair now
// owns a run of SP_NC cells (ix0 .. ix0 + NC - 1, ix0 a multiple of NC) and walks the union of their lists, (sample, one weight per
// cell): the same FMAs plus those with a zero weight, which leave the sum unchanged: the result is bit-identical to the per-cell
// form.  Lists are plan-time data as before; the first SP_NR entries stay in registers across the groups of the slab (the rest is
// re-read from L1 / L2 per block of groups).
#ifndef SP_NR_
#define SP_NR_ (SP_NC == 2 ? 4 : 6)      // 4 entries + four CTAs per SM (64 registers) measured 2.71 ms against 2.79 ms for 8 entries + three CTAs
#endif
constexpr int SP_NR = SP_NR_;                             // list entries kept in registers
constexpr int SP_RUNS = 256 / SP_NC;                      // runs per 32 x 8 tile
#ifndef SP_LB
#define SP_LB 4                        // CTAs per SM the main kernel is compiled for
#endif
struct SpW { float w[SP_NC]; };

template <class F>
__device__ __forceinline__ void enum_run_taps(const DevPlan &d, const TileRange *__restrict__ rng, const int *__restrict__ nrng,
                                              int tile, int ix0, int iy, F f) {
    const int G = d.G, nd = d.nd, na = d.na;
    const int Kx0 = ix0 < G / 2 ? ix0 : ix0 - G, Ky0 = iy < G / 2 ? iy : iy - G;      // cell c is Kx0 + c (a run never straddles G / 2)
    const int mmax = nd / 2 - 1, J = d.J;
    const int nr = nrng[tile];
    for (int e = 0; e < nr; ++e) {
        const TileRange tr = rng[tile * 4 + e];
        const int Kx = Kx0 + tr.shx, Ky = Ky0 + tr.shy;
        const float Kxf = (float)Kx, Kyf = (float)Ky, Kxl = Kxf + (float)(SP_NC - 1);
        for (int i = 0; i < tr.count; ++i) {
            int k = tr.start + i; if (k >= na) k -= na;
            const double2 cs = d.cs_sorted[k];
            const float cf = (float)cs.x, sf = (float)cs.y;
            const float acf = fabsf(cf), asf = fabsf(sf);
            // the ray misses the box of the whole run (the boxes of the cells, widened by the run's extent along x)
            if (fabsf((Kxf + 0.5f * (SP_NC - 1)) * sf - Kyf * cf) > d.hwf * (acf + asf) + 0.5f * (SP_NC - 1) * asf + 0.02f) continue;
            const float mc0 = acf >= asf ? Kxf / cf : Kyf / sf, mc1 = acf >= asf ? Kxl / cf : mc0;
            const int ma = __float2int_rn(fminf(mc0, mc1)) - J - 1, mb = __float2int_rn(fmaxf(mc0, mc1)) + J + 1;
            const int a = d.a_sorted[k];
            for (int m = max(ma, -mmax); m <= min(mb, mmax); ++m) {
                const double kx = __dmul_rn((double)m, cs.x), dy = __dmul_rn((double)m, cs.y) - Ky;       // rounded products (enum_cell_taps)
                if (dy <= -d.hw || dy > d.hw) continue;
                SpW w; bool any = false;
                const float wy = kb_eval(d, (float)dy);
#pragma unroll
                for (int c = 0; c < SP_NC; ++c) {
                    const double dx = kx - (Kx + c);
                    const bool in = dx > -d.hw && dx <= d.hw;
                    w.w[c] = in ? kb_eval(d, (float)dx) * wy : 0.f;
                    any = any || in;
                }
                if (any) f(a * nd + (m < 0 ? m + nd : m), w);
            }
        }
    }
}
// run q of a tile (the order of spread_cell): first cell c0, cells c0 .. c0 + NC - 1
__device__ __forceinline__ void spread_run(int q, int bx, int by, int &c0, int &ix0, int &iy) {
    constexpr int RPW = 32 / SP_NC;                       // runs per 32 cells of spread_cell's order
    const int cw = q / RPW, cl = (q % RPW) * SP_NC;
    c0 = cw * 32 + cl;
    ix0 = bx * 32 + (cw & 3) * 8 + (cl & 7); iy = by * 8 + (cw >> 2) * 4 + (cl >> 3);
}
__global__ void __launch_bounds__(SP_RUNS) k_run_count(DevPlan d, unsigned *__restrict__ counts) {
    int c0, ix0, iy; spread_run(threadIdx.x, blockIdx.x, blockIdx.y, c0, ix0, iy);
    const int tile = blockIdx.y * gridDim.x + blockIdx.x;
    unsigned n = 0;
    if (ix0 < d.G && iy < d.G) enum_run_taps(d, d.tile_rng, d.tile_nr, tile, ix0, iy, [&](int, const SpW &) { ++n; });
    counts[tile * SP_RUNS + threadIdx.x] = n;
}
__global__ void __launch_bounds__(SP_RUNS) k_run_fill(DevPlan d, const unsigned *__restrict__ poffs, int *__restrict__ pidx, SpW *__restrict__ pw) {
    int c0, ix0, iy; spread_run(threadIdx.x, blockIdx.x, blockIdx.y, c0, ix0, iy);
    const int tile = blockIdx.y * gridDim.x + blockIdx.x;
    if (ix0 >= d.G || iy >= d.G) return;
    unsigned o = poffs[tile * SP_RUNS + threadIdx.x];
    enum_run_taps(d, d.tile_rng, d.tile_nr, tile, ix0, iy, [&](int idx, const SpW &w) { pidx[o] = idx; pw[o] = w; ++o; });
}

template <int GPT>
__device__ __forceinline__ void run_tap(const float4 *__restrict__ cg, const size_t (&qoff)[GPT], int idx, const SpW &w, float4 (&acc)[SP_NC][GPT]) {
    const float4 *ca = cg + (size_t)idx * 2;
#pragma unroll
    for (int k = 0; k < GPT; ++k) {
        const float4 v = __ldg(ca + qoff[k]);
#pragma unroll
        for (int c = 0; c < SP_NC; ++c) {
            acc[c][k].x = fmaf(w.w[c], v.x, acc[c][k].x); acc[c][k].y = fmaf(w.w[c], v.y, acc[c][k].y);
            acc[c][k].z = fmaf(w.w[c], v.z, acc[c][k].z); acc[c][k].w = fmaf(w.w[c], v.w, acc[c][k].w);
        }
    }
}
__device__ __forceinline__ SpW spw_load(const SpW *p) {
    SpW w;
    if constexpr (SP_NC == 2) { const float2 t = __ldg(reinterpret_cast<const float2 *>(p)); w.w[0] = t.x; w.w[1] = t.y; }
    else { const float4 t = __ldg(reinterpret_cast<const float4 *>(p)); w.w[0] = t.x; w.w[1] = t.y; w.w[SP_NC - 2] = t.z; w.w[SP_NC - 1] = t.w; }
    return w;
}

template <int GPT>
__global__ void __launch_bounds__(2 * SP_RUNS, SP_LB) k_adj_spread_runs(DevPlan d, const unsigned *__restrict__ offs, const unsigned *__restrict__ poffs,
                                                            const int *__restrict__ pidx, const SpW *__restrict__ pw,
                                                            const float2 *__restrict__ cpol, int ng, float2 *__restrict__ grid) {
    const int q = threadIdx.x >> 1, hp = threadIdx.x & 1, G = d.G;
    int c0, ix0, iy; spread_run(q, blockIdx.x, blockIdx.y, c0, ix0, iy);
    if (ix0 >= G || iy >= G) return;
    const int tile = blockIdx.y * gridDim.x + blockIdx.x, cidx = tile * 256 + c0;
    const int R = d.discR, ks = iy < G / 2 ? iy : iy - G, kf0 = ix0 < G / 2 ? ix0 : ix0 - G;
    bool st[SP_NC], any = false;
    {
        unsigned o[SP_NC + 1];
#pragma unroll
        for (int c = 0; c <= SP_NC; ++c) o[c] = offs[cidx + c];
#pragma unroll
        for (int c = 0; c < SP_NC; ++c) {
            if (o[c + 1] - o[c] > SPREAD_HEAVY) return;              // the whole run goes to k_adj_spread_heavy (k_spread_heavy_list lists run mates)
            // a cell without taps outside the sampled disc is not written: nobody reads it (see disc_live)
            st[c] = o[c + 1] > o[c] || (kf0 + c) * (kf0 + c) + ks * ks <= R * R;
            any = any || st[c];
        }
    }
    if (!any) return;
    const unsigned t0 = poffs[tile * SP_RUNS + q], t1 = poffs[tile * SP_RUNS + q + 1];
    int ei[SP_NR]; SpW ew[SP_NR];                                        // entries past the end of the list: (sample 0, weights 0)
#pragma unroll
    for (int u = 0; u < SP_NR; ++u) {
        const bool in = t0 + u < t1;
        ei[u] = in ? __ldg(&pidx[t0 + u]) : 0;
        if (in) ew[u] = spw_load(&pw[t0 + u]);
        else {
#pragma unroll
            for (int c = 0; c < SP_NC; ++c) ew[u].w[c] = 0.f;
        }
    }
    const size_t gstride = (size_t)d.na * d.nd * 2, gg2 = (size_t)G * G * 2;
    // cell c of the run: parity block (c & 1), position (ix0 >> 1) + (c >> 1)
    float4 *out = reinterpret_cast<float4 *>(grid) + (((size_t)iy) * G + (ix0 >> 1)) * 2 + hp;
#pragma unroll 1
    for (int g0 = 0; g0 < ng; g0 += GPT) {
        float4 acc[SP_NC][GPT];
        size_t qoff[GPT];                                               // groups past the end re-read group g0 and are dropped at the store
#pragma unroll
        for (int k = 0; k < GPT; ++k) {
            qoff[k] = g0 + k < ng ? k * gstride : 0;
#pragma unroll
            for (int c = 0; c < SP_NC; ++c) acc[c][k] = make_float4(0.f, 0.f, 0.f, 0.f);
        }
        const float4 *cg = reinterpret_cast<const float4 *>(cpol) + (size_t)g0 * gstride + hp;
        if (t1 > t0) {
#pragma unroll
            for (int u = 0; u < SP_NR / 2; ++u) run_tap<GPT>(cg, qoff, ei[u], ew[u], acc);
        }
        if (t1 > t0 + SP_NR / 2) {
#pragma unroll
            for (int u = SP_NR / 2; u < SP_NR; ++u) run_tap<GPT>(cg, qoff, ei[u], ew[u], acc);
        }
        for (unsigned t = t0 + SP_NR; t < t1; ++t) run_tap<GPT>(cg, qoff, __ldg(&pidx[t]), spw_load(&pw[t]), acc);
#pragma unroll
        for (int k = 0; k < GPT; ++k)
            if (g0 + k < ng) {
#pragma unroll
                for (int c = 0; c < SP_NC; ++c)
                    if (st[c]) out[(size_t)(g0 + k) * gg2 + ((size_t)(c & 1) * (G >> 1) + (c >> 1)) * 2] = acc[c][k];
            }
    }
}

void launch_tile_ranges(const DevPlan &d, TileRange *rng, int *nrng, cudaStream_t st) {
    const int nt = ((d.G + 31) / 32) * ((d.G + 7) / 8);
    k_tile_ranges<<<(nt + 127) / 128, 128, 0, st>>>(d, rng, nrng);
}

// ------------------------------------------------------------------------------------------------
template <typename K> static void set_smem(K k, size_t bytes) {
    if (bytes > 48 * 1024) cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
}

#define TC_LINE_LAUNCH1(KERNEL, PLN, CFG, THR, fd, gr, ...)                          \
    do {                                                                        \
        const size_t sh = (size_t)(fd).smem_cells * PLN * sizeof(float2);       \
        set_smem(KERNEL<CFG>, sh);                                              \
        KERNEL<CFG><<<gr, (THR) ? (THR) : CFG::SLOTS * PLN, sh, st>>>(__VA_ARGS__); \
    } while (0)
// compile-time pass lists for the sizes of the BASELINE configs (must equal make_fft_desc's), run-time otherwise
#define TC_LINE_LAUNCH(KERNEL, PLN, TWS, THR, fd, gr, ...)                                                              \
    do {                                                                                                      \
        switch ((fd).n) {                                                                                     \
        case 256:  TC_LINE_LAUNCH1(KERNEL, PLN, TC_SC(PLN, 256, TWS, 16, 16), THR, fd, gr, __VA_ARGS__); break;              \
        case 1024: TC_LINE_LAUNCH1(KERNEL, PLN, TC_SC(PLN, 1024, TWS, 16, 16, 4), THR, fd, gr, __VA_ARGS__); break;          \
        case 2048: TC_LINE_LAUNCH1(KERNEL, PLN, TC_SC(PLN, 2048, TWS, 16, 16, 8), THR, fd, gr, __VA_ARGS__); break;          \
        case 2560: TC_LINE_LAUNCH1(KERNEL, PLN, TC_SC(PLN, 2560, TWS, 16, 16, 2, 5), THR, fd, gr, __VA_ARGS__); break;       \
        default:   TC_LINE_LAUNCH1(KERNEL, PLN, RCfgT<PLN>, THR, fd, gr, __VA_ARGS__); break;                                 \
        }                                                                                                     \
        TC_COUNT_LAUNCH();                                                                                    \
    } while (0)
#define TC_SC(...) SCfg<__VA_ARGS__>

static bool launch_fwd_rows_tma(const DevPlan &d, const float *vol, int S, int ng, float2 *rowbuf, cudaStream_t st);
static bool launch_adj_cols_tma(const DevPlan &d, const float2 *grid, int ng, float2 *rowbuf, cudaStream_t st);
static bool launch_adj_radial_tma(const DevPlan &d, const float *sino, int S, int ng, float2 *cpol, cudaStream_t st);
static bool env_is(const char *name, const char *value);
void launch_fwd_rows(const DevPlan &d, const float *vol, int S, int ng, float2 *rowbuf, cudaStream_t st) {
    static const bool plain = env_is("TC_FROWS", "plain");
    if (!plain && launch_fwd_rows_tma(d, vol, S, ng, rowbuf, st)) return;
    TC_LINE_LAUNCH(k_fwd_rows, 2, 2, 0, d.fN, dim3(2 * d.n, ng), d, vol, S, rowbuf);
}
static bool launch_fwd_cols_tma(const DevPlan &d, const float2 *rowbuf, int ng, float2 *grid, cudaStream_t st);   // kernels_line_tma.cuh
static bool env_is(const char *name, const char *value) { const char *e = std::getenv(name); return e && std::string(e) == value; }
void launch_fwd_cols(const DevPlan &d, const float2 *rowbuf, int ng, float2 *grid, cudaStream_t st) {
    static const bool plain = env_is("TC_COLS", "plain");
    if (!plain && launch_fwd_cols_tma(d, rowbuf, ng, grid, st)) return;
    TC_LINE_LAUNCH(k_fwd_cols, 4, 2, 0, d.fN, dim3(d.G, ng), d, rowbuf, grid);
}
void launch_adj_cols(const DevPlan &d, const float2 *grid, int ng, float2 *rowbuf, cudaStream_t st) {
    static const bool plain = env_is("TC_ACOLS", "plain");
    if (!plain && launch_adj_cols_tma(d, grid, ng, rowbuf, st)) return;
    TC_LINE_LAUNCH(k_adj_cols, 4, 2, 0, d.fN, dim3(d.G, ng), d, grid, rowbuf);
}
static bool launch_adj_rows_tma(const DevPlan &d, const float2 *rowbuf, int S, int ng, float *vol, cudaStream_t st);   // kernels_line_tma.cuh
void launch_adj_rows(const DevPlan &d, const float2 *rowbuf, int S, int ng, float *vol, cudaStream_t st) {
    static const bool plain = env_is("TC_AROWS", "plain");
    if (!plain && launch_adj_rows_tma(d, rowbuf, S, ng, vol, st)) return;
    TC_LINE_LAUNCH(k_adj_rows, 4, 2, 0, d.fN, dim3(d.n, ng), d, rowbuf, S, vol);
}
void launch_fwd_gather(const DevPlan &d, const float2 *grid, int S, int ng, float *sino, cudaStream_t st) {
    TC_LINE_LAUNCH(k_fwd_gather, 4, 1, GATHER_THREADS, d.fD, dim3(d.na, ng), d, grid, S, sino);
}
void launch_adj_radial(const DevPlan &d, const float *sino, int S, int ng, float2 *cpol, cudaStream_t st) {
    static const bool plain = env_is("TC_ARAD", "plain");
    if (!plain && launch_adj_radial_tma(d, sino, S, ng, cpol, st)) return;
    TC_LINE_LAUNCH(k_adj_radial, 4, 1, 0, d.fD, dim3(d.na, ng), d, sino, S, cpol);
}
void launch_spread_count(const DevPlan &d, int *counts, cudaStream_t st) {
    k_spread_count<<<dim3((d.G + 31) / 32, (d.G + 7) / 8), 256, 0, st>>>(d, d.tile_rng, d.tile_nr, counts);
}
void launch_spread_fill(const DevPlan &d, cudaStream_t st) {
    k_spread_fill<<<dim3((d.G + 31) / 32, (d.G + 7) / 8), 256, 0, st>>>(d, d.tile_rng, d.tile_nr, d.tap_offs, const_cast<int2 *>(d.taps));
}
int spread_run_cells() { return SP_NC; }
void launch_pair_count(const DevPlan &d, unsigned *counts, cudaStream_t st) {
    k_run_count<<<dim3((d.G + 31) / 32, (d.G + 7) / 8), SP_RUNS, 0, st>>>(d, counts);
}
void launch_pair_fill(const DevPlan &d, int *pidx, void *pw, cudaStream_t st) {
    k_run_fill<<<dim3((d.G + 31) / 32, (d.G + 7) / 8), SP_RUNS, 0, st>>>(d, d.pair_offs, pidx, static_cast<SpW *>(pw));
}
void launch_spread_heavy_list(const DevPlan &d, unsigned ncell, unsigned *list, unsigned *count, cudaStream_t st) {
    k_spread_heavy_list<<<(ncell + 255) / 256, 256, 0, st>>>(d, d.tap_offs, ncell, list, count);
}
void launch_adj_spread(const DevPlan &d, const float2 *cpol, int ng, float2 *grid, cudaStream_t st) {
    const int gpt = ng >= 4 ? 4 : (ng >= 2 ? 2 : 1), nz = (ng + gpt - 1) / gpt;
    // the heavy cells (long serial lists, few warps) run beside the main kernel on the plan's side stream: disjoint cells
    cudaStream_t hs = st;
    if (d.n_heavy && d.side) {
        cudaEventRecord(d.ev_fork, st);
        cudaStreamWaitEvent(d.side, d.ev_fork, 0);
        hs = d.side;
    }
    if (d.n_heavy) {
        const dim3 hg((d.n_heavy + 7) / 8, nz);
        if (gpt == 4) k_adj_spread_heavy<4><<<hg, 256, 0, hs>>>(d, d.tap_offs, d.taps, d.heavy, d.n_heavy, cpol, ng, grid);
        else if (gpt == 2) k_adj_spread_heavy<2><<<hg, 256, 0, hs>>>(d, d.tap_offs, d.taps, d.heavy, d.n_heavy, cpol, ng, grid);
        else k_adj_spread_heavy<1><<<hg, 256, 0, hs>>>(d, d.tap_offs, d.taps, d.heavy, d.n_heavy, cpol, ng, grid);
        TC_COUNT_LAUNCH();
        if (hs != st) cudaEventRecord(d.ev_join, hs);
    }
    const dim3 bl(512), gr((d.G + 31) / 32, (d.G + 7) / 8, 1);     // the group blocks are looped inside the kernel
    if (d.pair_offs && !env_is("TC_SPREAD", "plain")) {
        const SpW *pw = static_cast<const SpW *>(d.pair_w);
        if (ng >= 2) k_adj_spread_runs<2><<<gr, 2 * SP_RUNS, 0, st>>>(d, d.tap_offs, d.pair_offs, d.pair_idx, pw, cpol, ng, grid);
        else k_adj_spread_runs<1><<<gr, 2 * SP_RUNS, 0, st>>>(d, d.tap_offs, d.pair_offs, d.pair_idx, pw, cpol, ng, grid);
        TC_COUNT_LAUNCH();
        if (hs != st) cudaStreamWaitEvent(st, d.ev_join, 0);
        return;
    }
    if (gpt == 4) k_adj_spread<4><<<gr, bl, 0, st>>>(d, d.tap_offs, d.taps, cpol, ng, grid);
    else if (gpt == 2) k_adj_spread<2><<<gr, bl, 0, st>>>(d, d.tap_offs, d.taps, cpol, ng, grid);
    else k_adj_spread<1><<<gr, bl, 0, st>>>(d, d.tap_offs, d.taps, cpol, ng, grid);
    TC_COUNT_LAUNCH();
    if (hs != st) cudaStreamWaitEvent(st, d.ev_join, 0);
}
