// Line FFT engine: one CTA transforms one line of PL complex planes (PL = 4: whole 32-byte cells; PL = 2: 16-byte halves of
// them), length n = R1 R2 ... RL, with the first pass fused into the load and the last pass fused into the store.
//
// Thread t owns plane pl = t % PL and task slot t / PL (SLOTS * PL threads): with PL = 4 the four lanes of a quad touch the four
// 8-byte planes of the same 32-byte cell in the same instruction, so every global access is a whole sector.  A task is one
// radix-R butterfly of one plane, held in registers; tasks of a pass are independent, a thread runs any number
// of them one after the other, and there is one barrier per pass.
//
// Decimation in frequency with a transposing first pass, all later passes in place:
//   first pass   task b < n/R1:  x[b + (n/R1) j] (from `ld`)  -> DFT over j -> * w_n^{b k1} -> cell R1 b + k1
//   pass i       sub-transform of size n_i = n / (R1..R_{i-1}) inside every residue; task (outer, b_i, k1):
//                cells R1 (outer n_i + j_i (n_i/R_i) + b_i) + k1, j_i < R_i, DFT over j_i in place,
//                * w_{n_i}^{b_i k_i}
//   last pass    (n_L = R_L, no twiddles) task T = k1 + R1 k2 + ...: outputs X[T + (n/R_L) k_L] go to `st`
// Shared-memory cell c is stored at c + (c >> 4) (one padding cell per 16) so that the first pass's stride-R1
// writes and every later consecutive-k1 access are free of bank conflicts with 8-byte lanes.
// tw[i * tws] = e^{-2 pi i * i / n}.
#pragma once
#include "fft.cuh"

namespace tc {

constexpr int LINE_SLOTS = 128;               // most task slots per CTA; a CTA has Cfg::SLOTS * PL threads (PL = planes it carries: 4 or 2)
constexpr int LINE_THREADS = LINE_SLOTS * 4;    // the 4-plane form (polar kernels)

__device__ __forceinline__ int pcell(int c) { return c + (c >> 4); }

// Pass configuration: compile-time (every index, stride and radix folds to an immediate) for the sizes of the
// BASELINE configs, run-time (from the descriptor) for everything else.  TWS = stride of the twiddle table.
template <int PL_, int N_, int TWS_, int... Rs> struct SCfg {
    static constexpr bool is_static = true;
    static constexpr bool PM_LAST = false;
    static constexpr int GROUP_THREADS = 0;
    static constexpr int PL = PL_;
    static constexpr int SLOTS = N_ / 16 < LINE_SLOTS ? (N_ / 16 < 32 ? 32 : N_ / 16) : LINE_SLOTS;   // one radix-16 task per thread when the line is short
    static constexpr int NP = sizeof...(Rs);
    __device__ __forceinline__ static constexpr int n() { return N_; }
    __device__ __forceinline__ static constexpr int tws() { return TWS_; }
    __device__ __forceinline__ static constexpr int npass() { return NP; }
    __device__ __forceinline__ static constexpr int radix(int i) { constexpr int r[NP] = {Rs...}; return r[i]; }
};
template <int PL_> struct RCfgT {
    static constexpr bool is_static = false;
    static constexpr bool PM_LAST = false;
    static constexpr int GROUP_THREADS = 0;
    static constexpr int PL = PL_;
    static constexpr int SLOTS = LINE_SLOTS;
    FftDesc d; int tws_;
    __device__ __forceinline__ int n() const { return d.n; }
    __device__ __forceinline__ int tws() const { return tws_; }
    __device__ __forceinline__ int npass() const { return d.npass; }
    __device__ __forceinline__ int radix(int i) const { return d.radix[i]; }
};

// Plane-major last pass: thread = (plane, slot) instead of (slot, plane), so a warp's stores are 32 consecutive outputs of ONE
// plane (a full 128-byte line per float slice) -- for kernels whose output is the float volume.  In the [cell][plane] layout that
// pass's shared-memory reads have 4-way bank conflicts; the grouped kernels stage the data plane-major first (line_mid_pm).
template <class Base> struct PlaneMajorLast : Base { static constexpr bool PM_LAST = true; };

// Grouped form: a CTA holds several independent groups of GT threads (GT = SLOTS * PL), each transforming its own line in its own
// shared-memory buffer; the barrier between passes is the group's named barrier (1 + group index), not the CTA's.
template <class Base, int GT> struct Grouped : Base { static constexpr int GROUP_THREADS = GT; };
template <class Cfg> __device__ __forceinline__ int line_tid() {
    if constexpr (Cfg::GROUP_THREADS == 0) return threadIdx.x; else return threadIdx.x % Cfg::GROUP_THREADS;
}
template <class Cfg> __device__ __forceinline__ void line_sync() {
    if constexpr (Cfg::GROUP_THREADS == 0) __syncthreads();
    else asm volatile("bar.sync %0, %1;" ::"r"(1 + threadIdx.x / Cfg::GROUP_THREADS), "n"(Cfg::GROUP_THREADS) : "memory");
}

struct LineCtx {
    float2 *sm;               // [padded cell][4 planes]
    const float2 *tw;
    int pl, slot;
};

// v[k] *= w^k, w = tw[base * tws] (conjugated for the inverse); powers from tw[base], tw[2 base], tw[4 base], tw[8 base]
template <int R, bool INV>
__device__ __forceinline__ void twiddle_mul(const float2 *__restrict__ t, int e, float2 (&v)[R], int len = 0) {
    if constexpr ((R & 1) == 1) {                      // odd radix: one table entry per factor, exponent reduced modulo the table length
#pragma unroll
        for (int k = 1; k < R; ++k) {
            float2 w = __ldg(t + (k * e) % len);
            if (INV) w.y = -w.y;
            v[k] = cmul(v[k], w);
        }
        return;
    }
    float2 w1 = __ldg(t + e);
    if (INV) w1.y = -w1.y;
    v[1] = cmul(v[1], w1);
    if (R > 2) {
        float2 w2 = __ldg(t + 2 * e); if (INV) w2.y = -w2.y;
        const float2 w3 = cmul(w1, w2);
        v[2] = cmul(v[2], w2); v[3] = cmul(v[3], w3);
        if (R > 4) {
            float2 w4 = __ldg(t + 4 * e); if (INV) w4.y = -w4.y;
            const float2 w5 = cmul(w4, w1), w6 = cmul(w4, w2), w7 = cmul(w4, w3);
            v[4] = cmul(v[4], w4); v[5] = cmul(v[5], w5); v[6] = cmul(v[6], w6); v[7] = cmul(v[7], w7);
            if (R > 8) {
                float2 w8 = __ldg(t + 8 * e); if (INV) w8.y = -w8.y;
                v[8] = cmul(v[8], w8);
                v[9] = cmul(v[9], cmul(w8, w1)); v[10] = cmul(v[10], cmul(w8, w2)); v[11] = cmul(v[11], cmul(w8, w3));
                v[12] = cmul(v[12], cmul(w8, w4)); v[13] = cmul(v[13], cmul(w8, w5)); v[14] = cmul(v[14], cmul(w8, w6));
                v[15] = cmul(v[15], cmul(w8, w7));
            }
        }
    }
}

// first pass: global (through ld) -> shared
template <int R, bool INV, class Cfg, class LD>
__device__ __forceinline__ void line_first(const LineCtx &c, const Cfg &cfg, LD ld) {
    const int nb = cfg.n() / R;
#pragma unroll 1
    for (int b = c.slot; b < nb; b += Cfg::SLOTS) {
        float2 v[R];
#pragma unroll
        for (int j = 0; j < R; ++j) v[j] = ld(b + nb * j, R % 2 == 0 ? j < R / 2 : 2 * (b + nb * j) < cfg.n());
        Bfly<R, INV>::run(v);
        twiddle_mul<R, INV>(c.tw, b * cfg.tws(), v);
        float2 *o = c.sm + pcell(R * b) * Cfg::PL + c.pl;   // R b is a multiple of R and R divides 16: k never crosses a padding cell
#pragma unroll
        for (int k = 0; k < R; ++k) o[k * Cfg::PL] = v[k];
    }
    line_sync<Cfg>();
}

// first pass when the producer already left the line in shared memory: element t = b + (n/R) j at cell R b + j
// (line_input_cell), transformed in place.
__device__ __forceinline__ int line_input_cell(int n, int R1, int t) { const int nb = n / R1; const int j = t / nb; return pcell(R1 * (t - j * nb) + j); }

template <int R, bool INV, class Cfg>
__device__ __forceinline__ void line_first_smem(const LineCtx &c, const Cfg &cfg) {
    const int nb = cfg.n() / R;
#pragma unroll 1
    for (int b = c.slot; b < nb; b += Cfg::SLOTS) {
        float2 v[R];
        float2 *o = c.sm + pcell(R * b) * Cfg::PL + c.pl;
#pragma unroll
        for (int j = 0; j < R; ++j) v[j] = o[j * Cfg::PL];
        Bfly<R, INV>::run(v);
        twiddle_mul<R, INV>(c.tw, b * cfg.tws(), v);
#pragma unroll
        for (int k = 0; k < R; ++k) o[k * Cfg::PL] = v[k];
    }
    line_sync<Cfg>();
}

// first pass when the raw line sits in the SAME buffer in some other layout (brought in by TMA): every thread takes its R inputs
// into registers (through ld), a barrier lets the whole line leave shared memory, then the results go to the work layout.
// One task per thread: n / R == SLOTS.
template <int R, bool INV, class Cfg, class LD>
__device__ __forceinline__ void line_first_inplace(const LineCtx &c, const Cfg &cfg, LD ld) {
    static_assert(Cfg::is_static, "compile-time pass list only");
    constexpr int nb = Cfg::n() / R;
    static_assert(nb == Cfg::SLOTS, "one first-pass task per thread");
    const int b = c.slot;
    float2 v[R];
    if (b < nb) {
#pragma unroll
        for (int j = 0; j < R; ++j) v[j] = ld(b + nb * j, R % 2 == 0 ? j < R / 2 : 2 * (b + nb * j) < cfg.n());
    }
    line_sync<Cfg>();
    if (b < nb) {
        Bfly<R, INV>::run(v);
        twiddle_mul<R, INV>(c.tw, b * cfg.tws(), v);
        float2 *o = c.sm + pcell(R * b) * Cfg::PL + c.pl;
#pragma unroll
        for (int k = 0; k < R; ++k) o[k * Cfg::PL] = v[k];
    }
    line_sync<Cfg>();
}

// pass i (not the last): in place.  s = R1 .. R_{i-1}, ni = n / s.
template <int R, bool INV, class Cfg>
__device__ __forceinline__ void line_mid(const LineCtx &c, const Cfg &cfg, int s) {
    const int n = cfg.n(), R1 = cfg.radix(0);
    const int ni = n / s, sub = ni / R;                 // sub = n_i / R_i = range of b_i
    const int ntask = n / R;
    const bool fast = ((R1 * sub) & 15) == 0;
    const int step = pcell(R1 * sub) * Cfg::PL;
#pragma unroll 1
    for (int T = c.slot; T < ntask; T += Cfg::SLOTS) {
        const int k1 = T % R1, rest = T / R1;
        const int outer = rest / sub, bi = rest - outer * sub;
        const int c0 = R1 * (outer * ni + bi) + k1;
        float2 v[R];
        float2 *p0 = c.sm + pcell(c0) * Cfg::PL + c.pl;
        if (fast) {
#pragma unroll
            for (int j = 0; j < R; ++j) v[j] = p0[j * step];
        } else {
#pragma unroll
            for (int j = 0; j < R; ++j) v[j] = c.sm[pcell(c0 + j * R1 * sub) * Cfg::PL + c.pl];
        }
        Bfly<R, INV>::run(v);
        twiddle_mul<R, INV>(c.tw, bi * s * cfg.tws(), v, n * cfg.tws());
        if (fast) {
#pragma unroll
            for (int j = 0; j < R; ++j) p0[j * step] = v[j];
        } else {
#pragma unroll
            for (int j = 0; j < R; ++j) c.sm[pcell(c0 + j * R1 * sub) * Cfg::PL + c.pl] = v[j];
        }
    }
    line_sync<Cfg>();
}

// last pass: shared -> global (through st).  Task T = k1 + R1 (k2 + R2 (k3 + ...)) < n / R, so that the R outputs
// X[T + (n/R) k] of consecutive tasks are consecutive; the middle digits k2.. sit in shared memory in position
// order (k2 most significant), hence the digit walk.
// pre(k, lo) is called for the task's R outputs before the butterfly (a read-modify-write caller starts its loads
// there) and its value is handed to st(k, lo, v, old).  lo = "k < n / 2", a compile-time fact for even radices.
struct NoPre { __device__ __forceinline__ float2 operator()(int, bool) const { return make_float2(0.f, 0.f); } };

template <int R, bool INV, class Cfg, class PRE, class ST>
__device__ __forceinline__ void line_last(const LineCtx &c, const Cfg &cfg, PRE pre, ST st) {
    const int n = cfg.n(), R1 = cfg.radix(0), ntask = n / R;
    const bool fast = (R1 & 15) == 0;
    const int step = pcell(R1) * Cfg::PL;
    const int my_pl = Cfg::PM_LAST ? line_tid<Cfg>() / Cfg::SLOTS : c.pl, my_slot = Cfg::PM_LAST ? line_tid<Cfg>() % Cfg::SLOTS : c.slot;
#pragma unroll 1
    for (int T = my_slot; T < ntask; T += Cfg::SLOTS) {
        const int k1 = T % R1;
        int rem = T / R1, mult = n / R1, B0 = 0;
#pragma unroll
        for (int i = 1; i + 1 < cfg.npass(); ++i) {
            const int Ri = cfg.radix(i);
            mult /= Ri;
            const int q = rem / Ri;
            B0 += (rem - q * Ri) * mult;
            rem = q;
        }
        const int c0 = R1 * B0 + k1;
        float2 v[R], old[R];
#pragma unroll
        for (int k = 0; k < R; ++k) old[k] = pre(T + ntask * k, R % 2 == 0 ? k < R / 2 : 2 * (T + ntask * k) < n);
        if (fast) {
            const float2 *p0 = c.sm + pcell(c0) * Cfg::PL + my_pl;
#pragma unroll
            for (int j = 0; j < R; ++j) v[j] = p0[j * step];
        } else {
#pragma unroll
            for (int j = 0; j < R; ++j) v[j] = c.sm[pcell(c0 + j * R1) * Cfg::PL + my_pl];
        }
        Bfly<R, INV>::run(v);
#pragma unroll
        for (int k = 0; k < R; ++k) st(T + ntask * k, R % 2 == 0 ? k < R / 2 : 2 * (T + ntask * k) < n, v[k], old[k]);
    }
}

// Plane-major staging for the plane-major last pass (PM_LAST): the last in-place pass leaves its results as [plane][cell] (plane
// stride n + 8 cells, no padding cells) instead of [cell][plane], so that the last pass -- a warp = 32 consecutive tasks of ONE
// plane -- reads consecutive 8-byte words (two wavefronts per instruction) instead of every fourth (eight).  The layout change is not
// in place, so the pass reads, meets the group's barrier, then writes: one task per thread (n / R == SLOTS).
template <class Cfg> __device__ __forceinline__ constexpr int pm_stride() { return Cfg::n() + 8; }
template <int R, bool INV, class Cfg>
__device__ __forceinline__ void line_mid_pm(const LineCtx &c, const Cfg &cfg, int s) {
    constexpr int n = Cfg::n(), R1 = Cfg::radix(0);
    static_assert(n / R == Cfg::SLOTS, "one task per thread");
    const int ni = n / s, sub = ni / R;
    const int T = c.slot;
    const bool on = T < n / R;
    float2 v[R];
    int c0 = 0;
    if (on) {
        const int k1 = T % R1, rest = T / R1;
        const int outer = rest / sub, bi = rest - outer * sub;
        c0 = R1 * (outer * ni + bi) + k1;
#pragma unroll
        for (int j = 0; j < R; ++j) v[j] = c.sm[pcell(c0 + j * R1 * sub) * Cfg::PL + c.pl];
        Bfly<R, INV>::run(v);
        twiddle_mul<R, INV>(c.tw, bi * s * cfg.tws(), v, n * cfg.tws());
    }
    line_sync<Cfg>();                                   // every task has its inputs: the buffer may change layout
    if (on) {
        float2 *o = c.sm + c.pl * pm_stride<Cfg>() + c0;
#pragma unroll
        for (int j = 0; j < R; ++j) o[j * R1 * sub] = v[j];
    }
    line_sync<Cfg>();
}
template <int R, bool INV, class Cfg, class PRE, class ST>
__device__ __forceinline__ void line_last_pm(const LineCtx &c, const Cfg &cfg, PRE pre, ST st) {
    constexpr int n = Cfg::n(), R1 = Cfg::radix(0), ntask = n / R;
    const int my_pl = line_tid<Cfg>() / Cfg::SLOTS, my_slot = line_tid<Cfg>() % Cfg::SLOTS;
#pragma unroll 1
    for (int T = my_slot; T < ntask; T += Cfg::SLOTS) {
        const int k1 = T % R1;
        int rem = T / R1, mult = n / R1, B0 = 0;
#pragma unroll
        for (int i = 1; i + 1 < cfg.npass(); ++i) {
            const int Ri = cfg.radix(i);
            mult /= Ri;
            const int q = rem / Ri;
            B0 += (rem - q * Ri) * mult;
            rem = q;
        }
        const float2 *p0 = c.sm + my_pl * pm_stride<Cfg>() + R1 * B0 + k1;
        float2 v[R], old[R];
#pragma unroll
        for (int k = 0; k < R; ++k) old[k] = pre(T + ntask * k, R % 2 == 0 ? k < R / 2 : 2 * (T + ntask * k) < n);
#pragma unroll
        for (int j = 0; j < R; ++j) v[j] = p0[j * R1];
        Bfly<R, INV>::run(v);
#pragma unroll
        for (int k = 0; k < R; ++k) st(T + ntask * k, R % 2 == 0 ? k < R / 2 : 2 * (T + ntask * k) < n, v[k], old[k]);
    }
}

template <class Cfg>
__device__ __forceinline__ LineCtx line_ctx(float2 *sm, const float2 *tw) {
    LineCtx c;
    const int tid = line_tid<Cfg>();
    c.sm = sm; c.tw = tw; c.pl = tid % Cfg::PL;
    c.slot = tid < Cfg::SLOTS * Cfg::PL ? tid / Cfg::PL : (1 << 30);      // a CTA may have more threads (the gather): they only meet the barriers
    return c;
}

// ---- drivers: compile-time pass list ------------------------------------------------------------------
template <bool INV, class Cfg, int I, int S_, class PRE, class ST>
__device__ __forceinline__ void static_finish(const LineCtx &c, const Cfg &cfg, PRE pre, ST st) {
    constexpr int R = Cfg::radix(I);
    if constexpr (I + 1 < Cfg::NP) {
        if constexpr (I + 2 == Cfg::NP && Cfg::PM_LAST && Cfg::GROUP_THREADS != 0 && Cfg::n() / R == Cfg::SLOTS) line_mid_pm<R, INV>(c, cfg, S_);
        else line_mid<R, INV>(c, cfg, S_);
        static_finish<INV, Cfg, I + 1, S_ * R>(c, cfg, pre, st);
    } else {
        if constexpr (Cfg::PM_LAST && Cfg::GROUP_THREADS != 0 && I >= 2) {      // the grouped (TMA-fed) kernels only: the plain ones lose more on the extra barrier (2.48 -> 2.98 ms)
            if constexpr (Cfg::n() / Cfg::radix(I - 1) == Cfg::SLOTS) line_last_pm<R, INV>(c, cfg, pre, st);
            else line_last<R, INV>(c, cfg, pre, st);
        } else line_last<R, INV>(c, cfg, pre, st);
    }
}

// ---- drivers: run-time pass list ----------------------------------------------------------------------
template <bool INV, class Cfg, class PRE, class ST>
__device__ __forceinline__ void runtime_finish(const LineCtx &c, const Cfg &cfg, PRE pre, ST st) {
    int s = cfg.radix(0);
#pragma unroll 1
    for (int i = 1; i + 1 < cfg.npass(); ++i) {
        const int R = cfg.radix(i);
        if (R == 16) line_mid<16, INV>(c, cfg, s);
        else if (R == 8) line_mid<8, INV>(c, cfg, s);
        else if (R == 4) line_mid<4, INV>(c, cfg, s);
        else if (R == 2) line_mid<2, INV>(c, cfg, s);
        else if (R == 3) line_mid<3, INV>(c, cfg, s);
        else if (R == 5) line_mid<5, INV>(c, cfg, s);
        else if (R == 7) line_mid<7, INV>(c, cfg, s);
        else line_mid<17, INV>(c, cfg, s);
        s *= R;
    }
    const int RL = cfg.radix(cfg.npass() - 1);
    if (RL == 16) line_last<16, INV>(c, cfg, pre, st);
    else if (RL == 8) line_last<8, INV>(c, cfg, pre, st);
    else if (RL == 5) line_last<5, INV>(c, cfg, pre, st);
    else if (RL == 4) line_last<4, INV>(c, cfg, pre, st);
    else if (RL == 2) line_last<2, INV>(c, cfg, pre, st);
    else if (RL == 3) line_last<3, INV>(c, cfg, pre, st);
    else if (RL == 7) line_last<7, INV>(c, cfg, pre, st);
    else line_last<17, INV>(c, cfg, pre, st);
}

// global -> FFT -> global.  ld(t, lo) returns this thread's plane of input element t; st(k, lo, v, old) takes output k.
// A barrier must separate two transforms that use the same shared memory (the caller's job).
template <bool INV, class Cfg, class LD, class PRE, class ST>
__device__ __forceinline__ void fft_line(float2 *sm, const Cfg &cfg, const float2 *tw, LD ld, PRE pre, ST st) {
    const LineCtx c = line_ctx<Cfg>(sm, tw);
    if constexpr (Cfg::is_static) {
        line_first<Cfg::radix(0), INV>(c, cfg, ld);
        static_finish<INV, Cfg, 1, Cfg::radix(0)>(c, cfg, pre, st);
    } else {
        const int R1 = cfg.radix(0);
        if (R1 == 16) line_first<16, INV>(c, cfg, ld);
        else if (R1 == 8) line_first<8, INV>(c, cfg, ld);
        else if (R1 == 4) line_first<4, INV>(c, cfg, ld);
        else line_first<2, INV>(c, cfg, ld);
        runtime_finish<INV>(c, cfg, pre, st);
    }
}

// shared (filled at line_input_cell positions and synchronised by the caller) -> FFT -> global.
template <bool INV, class Cfg, class ST>
__device__ __forceinline__ void fft_line_from_smem(float2 *sm, const Cfg &cfg, const float2 *tw, ST st) {
    const LineCtx c = line_ctx<Cfg>(sm, tw);
    if constexpr (Cfg::is_static) {
        line_first_smem<Cfg::radix(0), INV>(c, cfg);
        static_finish<INV, Cfg, 1, Cfg::radix(0)>(c, cfg, NoPre(), st);
    } else {
        const int R1 = cfg.radix(0);
        if (R1 == 16) line_first_smem<16, INV>(c, cfg);
        else if (R1 == 8) line_first_smem<8, INV>(c, cfg);
        else if (R1 == 4) line_first_smem<4, INV>(c, cfg);
        else line_first_smem<2, INV>(c, cfg);
        runtime_finish<INV>(c, cfg, NoPre(), st);
    }
}

}  // namespace tc
