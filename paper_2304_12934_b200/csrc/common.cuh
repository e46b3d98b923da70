// Shared declarations of the tomoCAM B200 library (device-side plan view, launch wrappers).
#pragma once
#include <cuda_runtime.h>
#include "fft.cuh"

namespace tc {

constexpr int KB_W = 6;          // default Kaiser-Bessel window width (taps per axis); plans take 4, 6 or 8 (DevPlan::W)
constexpr int KB_DEG = 12;       // degree of the window polynomial in z = 2 q - 1, q = 1 - (2 r / W)^2
constexpr unsigned SPREAD_HEAVY = 96;   // tap lists longer than this are handled by one warp per cell (k_adj_spread_heavy)
#ifndef SP_NC
#define SP_NC 2                 // cells of a run of the spread (k_adj_spread_runs): 2 or 4
#endif
constexpr int P = 4;             // complex planes interleaved per fine-grid cell (= 8 real slices, 32 B)

struct TileRange { int start, count, shx, shy; };   // angles (sorted order) whose ray can touch a 32 x 8 tile, per wrap alias

// Everything the kernels need, passed by value.
struct DevPlan {
    int n, nd, na, G;
    int W;                        // window width (taps per axis): 4, 6 or 8; hw = W / 2
    double hw; float hwf;
    int discR;                    // fine-grid cells farther than this from the origin are never touched: G / 2 + W - 1
    float kb[KB_DEG + 1], kbs;    // window polynomial (monomial in z, c[0] + c[1] z + ...) and -2 / (W/2)^2: z = 1 - 2 (r / (W/2))^2; per plan
    double sc;                    // G / nd: fine-grid cells per radial mode
    FftDesc fN, fD;               // FFT descriptors for length n (half of the fine grid: pruned split) and nd (radial)
    const float2 *twG, *twD;      // twiddles e^{-2 pi i k / G} (length G; the length-n transforms use every 2nd) and e^{-2 pi i k / nd}
    const float *deapod;          // d(x_j) = 1 / phihat(x_j), j < n
    const float2 *ph_fwd;         // [nd] e^{-2 pi i m centre / nd} / nd, Nyquist entry 0 (forward, before the inverse radial FFT)
    const float2 *ph_adj;         // [nd] e^{+2 pi i m centre / nd} / nd, Nyquist entry 0 (adjoint, after the radial FFT)
    const double2 *cs;            // [na] (sc cos theta_a, sc sin theta_a)
    const double2 *cs_sorted;     // [na] same, sorted by theta mod pi
    const float *th_sorted;       // [na] theta mod pi, ascending
    const int *a_sorted;          // [na] original angle index
    const TileRange *tile_rng;    // [tiles][4]
    const int *tile_nr;           // [tiles] number of valid ranges
    const unsigned *tap_offs;     // [tiles * 256 + 1] CSR offsets of the spread's per-cell tap lists (cell order: tile, then thread)
    const int2 *taps;             // (a * nd + (m mod nd), float weight bits)
    const unsigned *pair_offs;    // [tiles * runs per tile + 1] CSR offsets of the lists of the cell runs (k_adj_spread_runs)
    const int *pair_idx;          // a * nd + (m mod nd)
    const void *pair_w;           // one weight per cell of the run (SpW)
    const unsigned *heavy;        // [n_heavy] cells (cidx) whose list, or whose pair partner's, is longer than SPREAD_HEAVY
    unsigned n_heavy;
    cudaStream_t side;            // the heavy-cell kernel runs beside the main spread kernel (disjoint cells): fork / join events
    cudaEvent_t ev_fork, ev_join;
    int J;                        // radial modes to try on each side of the nearest one: floor(3 sqrt2 / sc + 1/2)
    // tile-binned forward gather (k_fwd_gather_tiles): polar samples sorted by the fine-grid tile that holds their first tap
    int gt_ntx, gt_nty;           // tiles along the fast / slow axis
    int gt_nlive;                 // tiles that hold at least one sample
    int gt_nh, gt_nm;             // ranks [0, gt_nh): one group per work item, [gt_nh, gt_nm): four, the rest: sixteen
    const int *gt_tiles;          // [gt_nlive] tile ids (ty * gt_ntx + tx), most samples first
    const unsigned *gt_start;     // [gt_ntx gt_nty + 1] offsets into gt_samples
    const int4 *gt_samples;       // {a * nd + (m mod nd), (local base row << 16) | local base column, float bits of rx, of ry}
};

// Tile geometry of the binned gather: a tile owns the samples whose first tap (bx, by) falls into a GT_BX x GT_BY block of
// fine-grid cells (x = the grid's fast, parity-split axis) and stages GT_CX x GT_CY cells (block + the W - 1 = 5 cells the
// taps reach beyond it, rounded up to even) in shared memory, GT_NBUF tiles deep (GtDim<W>).
#ifndef GT_BX
#define GT_BX 90
#endif
#ifndef GT_BY
#define GT_BY 26
#endif
#ifndef GT_NBUF
#define GT_NBUF 2
#endif
template <int W> struct GtDim { static constexpr int CX = (GT_BX + W - 1 + 1) / 2 * 2, CY = GT_BY + W - 1; };
static_assert(GT_BX % 2 == 0, "tile origins must keep the parity of the fast axis");
__host__ __device__ inline int gt_pad(int W) { return (W / 2 + 1) & ~1; }      // first taps lie in [-G/2 - W/2, G/2 - W/2]; tile 0 starts on an even cell
__host__ __device__ inline int gt_min(int G, int W) { return -G / 2 - gt_pad(W); }   // centred coordinate of tile 0's first cell (even)
__host__ __device__ inline int gt_ntx(int G, int W) { return (G + 2 * gt_pad(W) + GT_BX - 1) / GT_BX; }
__host__ __device__ inline int gt_nty(int G, int W) { return (G + 2 * gt_pad(W) + GT_BY - 1) / GT_BY; }

// Roots of unity of the odd FFT radices (constant memory), set by the plan.
void set_fft_roots();

// ---- launch wrappers (kernels_nufft.cu).  All buffers are device memory. -------------------------
// vol [S][n][n] -> rowbuf [ng][n][G][P] c64      (F1 pad + deapodise, row FFT)
void launch_fwd_rows(const DevPlan &d, const float *vol, int S, int ng, float2 *rowbuf, cudaStream_t st);
// rowbuf -> grid [ng][G][G][P] c64               (F2 column FFT, zero rows pruned on input)
void launch_fwd_cols(const DevPlan &d, const float2 *rowbuf, int ng, float2 *grid, cudaStream_t st);
// grid -> sino [S][na][nd]                       (F3 polar gather + F4 centre phase and inverse radial FFT)
void launch_fwd_gather(const DevPlan &d, const float2 *grid, int S, int ng, float *sino, cudaStream_t st);
// tile-binned form of F3 (+ F4 as its own launch): grid -> cpol [ng][na][nd][P] c64 -> sino
void launch_gt_keys(const DevPlan &d, unsigned long long *keys, cudaStream_t st);
void launch_gt_fill(const DevPlan &d, const unsigned long long *keys, unsigned nvalid, int4 *samples, unsigned *counts, cudaStream_t st);
void launch_fwd_gather_tiles(const DevPlan &d, const float2 *grid, int ng, float2 *cpol, cudaStream_t st);
void launch_fwd_radial(const DevPlan &d, const float2 *cpol, int S, int ng, float *sino, cudaStream_t st);
// sino -> cpol [ng][na][nd][P] c64               (B1 radial FFT + conjugate phase)
void launch_adj_radial(const DevPlan &d, const float *sino, int S, int ng, float2 *cpol, cudaStream_t st);
// cpol -> grid                                   (B2 spread, evaluated per fine-grid cell: plain stores, no atomics)
void launch_tile_ranges(const DevPlan &d, TileRange *rng, int *nrng, cudaStream_t st);
void launch_spread_count(const DevPlan &d, int *counts, cudaStream_t st);
void launch_spread_fill(const DevPlan &d, cudaStream_t st);
void launch_spread_heavy_list(const DevPlan &d, unsigned ncell, unsigned *list, unsigned *count, cudaStream_t st);
void launch_pair_count(const DevPlan &d, unsigned *counts, cudaStream_t st);
void launch_pair_fill(const DevPlan &d, int *pidx, void *pw, cudaStream_t st);
int spread_run_cells();               // cells per run (2 or 4)
void launch_adj_spread(const DevPlan &d, const float2 *cpol, int ng, float2 *grid, cudaStream_t st);
// grid -> rowbuf (cropped to n rows)             (B3 inverse column FFT)
void launch_adj_cols(const DevPlan &d, const float2 *grid, int ng, float2 *rowbuf, cudaStream_t st);
// rowbuf -> vol (cropped, deapodised, re/im)     (B3 inverse row FFT + B4)
void launch_adj_rows(const DevPlan &d, const float2 *rowbuf, int S, int ng, float *vol, cudaStream_t st);

// ---- kernels_mbir.cu -------------------------------------------------------------------------------
struct PriorDev { float p, sigma, c, lambda; int nonneg = 0; int nbr = 26; };   // nbr: neighbour set of eq. (12): 26 (paper), 10 or 6
// y = x + beta (x - xm)                          (M1, volume part; only the streamed loop stores y)
void launch_extrapolate(const float *x, const float *xm, float beta, float *y, size_t n, cudaStream_t st);
// r = (Ax + beta (Ax - Axm)) - b                  (M1, sinogram part: A y is formed on the fly)
void launch_residual(const float *Ax, const float *Axm, const float *b, float beta, float *r, size_t n, cudaStream_t st);
// g = atr + lambda grad H(y);  z = y - g / L      (M2 + M3), y = x + beta (x - xm) formed on load (xm == nullptr: y = x).
// g may alias atr; z == nullptr: gradient only.  y has S slices; outputs are written for slices [s_first, s_first + n_out) only
// (n_out < 0: to the end) -- slabs with halos
void launch_update(const float *x, const float *xm, float beta, const float *atr, PriorDev pr, float invL, float *g, float *z, int S, int n,
                   cudaStream_t st, int s_first = 0, int n_out = -1);
// z = y - alpha g (projected on z >= 0 if nonneg), y as above     (candidate of the majorise-minimise step)
void launch_step(const float *x, const float *xm, float beta, const float *g, float alpha, int nonneg, float *z, size_t n, cudaStream_t st);
// Az = Ay - alpha Ag, Ay = A0 + beta (A0 - A1) (A1 == nullptr: Ay = A0; Ag == nullptr: Az = Ay);  acc[0] += 1/2 ||Az - b||^2   (M4 data term)
// rnext (nullable; may alias Ag): the next iteration's residual if the candidate is accepted, Az + beta_next (Az - A0) - b (A0 must be A x)
void launch_candidate_sino(const float *A0, const float *A1, const float *Ag, const float *b, float beta, float alpha, float *Az, double *acc,
                           size_t n, cudaStream_t st, float *rnext = nullptr, float beta_next = 0.f);
// acc[1] += H(z) over unordered neighbour pairs (M4 prior term); grad (nullable) = grad H(z)
// pairs are owned by their lower slice; only owners among the first S_own slices are summed (S_own < 0: all)
void launch_prior(const float *z, PriorDev pr, float *grad, double *acc, int S, int n, cudaStream_t st, int S_own = -1);
// acc[slot] += sum over pairs of w h'(D)/D (g_m - g_n)^2, D = y_m - y_n, y = x + beta (x - xm)   (surrogate curvature along g)
void launch_prior_curvature(const float *x, const float *xm, float beta, const float *g, PriorDev pr, double *acc, int slot, int S, int n, cudaStream_t st);
// acc[slot] += sum v^2
void launch_sumsq(const float *v, size_t n, double *acc, int slot, cudaStream_t st);
// acc[slot] += sum g (z - x)   (gradient restart test)
void launch_dot_gzx(const float *g, const float *z, const float *x, size_t n, double *acc, int slot, cudaStream_t st);
void launch_scale(float *v, float a, size_t n, cudaStream_t st);
// sino[s][a][u] = -log(max((proj[a][s][u] - dark[s][u]) / (flat[s][u] - dark[s][u]), floor))   (Beer-Lambert + reorder)
void launch_preprocess(const float *proj, const float *flat, const float *dark, int na, int S, int nd, float floor_, float *sino, cudaStream_t st);

// test hooks (tc_stage_*): one complex plane of group 0 in natural order <-> the internal layouts
void launch_grid_plane(float2 *grid, float2 *nat, int G, int pl, bool put, cudaStream_t st);
void launch_cpol_plane(float2 *cpol, float2 *nat, size_t n, int pl, bool put, cudaStream_t st);

long long &launch_counter();

}  // namespace tc

#define TC_COUNT_LAUNCH() (++::tc::launch_counter())
