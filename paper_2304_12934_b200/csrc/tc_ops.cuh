// Included by tc_api.cu: slab scheduler (S1), the public operator calls, the prior test hook, the in-core MBIR loop (M1-M5).

// Transfer / compute overlap of a streamed call, from the summed CUDA-event spans of its three streams (each stream is serial,
// so every busy time is <= wall): the part of the two shorter resources' work that was hidden behind the others,
//   overlap = (h2d + compute + d2h - wall) / (h2d + compute + d2h - max(h2d, compute, d2h))   in [0, 1];
// 1 = the wall time is the busiest resource's time alone, 0 = the three ran one after the other.
static double overlap_fraction(double h2d, double comp, double d2h, double wall) {
    const double sum = h2d + comp + d2h, mx = std::max(h2d, std::max(comp, d2h));
    if (sum - mx <= 0.0) return 0.0;
    return std::min(1.0, std::max(0.0, (sum - wall) / (sum - mx)));
}

static tc_status ensure_streams(tc_plan *p) {
    if (!p->s_h2d) {
        CU(cudaStreamCreateWithFlags(&p->s_h2d, cudaStreamNonBlocking));
        CU(cudaStreamCreateWithFlags(&p->s_comp, cudaStreamNonBlocking));
        CU(cudaStreamCreateWithFlags(&p->s_d2h, cudaStreamNonBlocking));
    }
    return TC_OK;
}

// Per-slab CUDA events of a streamed call (6 per slab: h2d, compute, d2h start / stop), destroyed on every return path.
struct SlabEvents {
    std::vector<cudaEvent_t> ev;
    cudaError_t create(size_t n) {
        ev.assign(n, nullptr);
        for (auto &e : ev) { cudaError_t r = cudaEventCreate(&e); if (r != cudaSuccess) return r; }
        return cudaSuccess;
    }
    cudaEvent_t *slab(int k) { return &ev[(size_t)k * 6]; }
    tc_status accumulate(int nslab, tc_sched_stats &st) {
        for (int k = 0; k < nslab; ++k) {
            float ms;
            CU(cudaEventElapsedTime(&ms, ev[(size_t)k * 6 + 0], ev[(size_t)k * 6 + 1])); st.h2d_s += ms * 1e-3;
            CU(cudaEventElapsedTime(&ms, ev[(size_t)k * 6 + 2], ev[(size_t)k * 6 + 3])); st.compute_s += ms * 1e-3;
            CU(cudaEventElapsedTime(&ms, ev[(size_t)k * 6 + 4], ev[(size_t)k * 6 + 5])); st.d2h_s += ms * 1e-3;
        }
        return TC_OK;
    }
    ~SlabEvents() { for (auto &e : ev) if (e) cudaEventDestroy(e); }
};

// ---- S1 slab scheduler: host-resident data streamed through device staging buffers (Fig. 3) ----
// Three streams (H2D, compute, D2H), two staging buffers per direction.  Slab k uses buffer k & 1:
//   H2D(k) waits compute(k-2) [input buffer free];  compute(k) waits H2D(k) and D2H(k-2) [output buffer free];
//   D2H(k) waits compute(k).  Slabs are views into the caller's arrays: nothing is repacked.
// Pageable caller memory is page-locked for the duration of the call (cudaHostRegister), otherwise its copies would be
// staged by the driver and serialise with everything else; if locking fails the call still runs, without overlap.
typedef void (*slab_op)(tc_plan *, const float *, int, float *, cudaStream_t);

static tc_status run_streamed(tc_plan *p, slab_op op, const float *hin, size_t in_per_slice, float *hout, size_t out_per_slice,
                              int S, int slab) {
    TCS(ensure_streams(p));
    const size_t need_in = (size_t)slab * in_per_slice, need_out = (size_t)slab * out_per_slice;
    if (p->stage_in_elems < need_in) {
        for (int b = 0; b < 2; ++b) { cudaFree(p->stage_in[b]); p->stage_in[b] = nullptr; }
        p->stage_in_elems = 0;
        for (int b = 0; b < 2; ++b) CU(cudaMalloc((void **)&p->stage_in[b], need_in * sizeof(float)));
        p->stage_in_elems = need_in;
    }
    if (p->stage_out_elems < need_out) {
        for (int b = 0; b < 2; ++b) { cudaFree(p->stage_out[b]); p->stage_out[b] = nullptr; }
        p->stage_out_elems = 0;
        for (int b = 0; b < 2; ++b) CU(cudaMalloc((void **)&p->stage_out[b], need_out * sizeof(float)));
        p->stage_out_elems = need_out;
    }
    CallMem mem;
    mem.pin(hin, (size_t)S * in_per_slice * sizeof(float));
    mem.pin(hout, (size_t)S * out_per_slice * sizeof(float));
    const int nslab = (S + slab - 1) / slab;
    SlabEvents evs;
    CU(evs.create((size_t)nslab * 6));
    auto t0 = std::chrono::steady_clock::now();
    for (int k = 0; k < nslab; ++k) {
        const int b = k & 1, s0 = k * slab, ns = std::min(slab, S - s0);
        cudaEvent_t *e = evs.slab(k);
        if (k >= 2) CU(cudaStreamWaitEvent(p->s_h2d, evs.slab(k - 2)[3], 0));
        CU(cudaEventRecord(e[0], p->s_h2d));
        CU(cudaMemcpyAsync(p->stage_in[b], hin + (size_t)s0 * in_per_slice, (size_t)ns * in_per_slice * sizeof(float), cudaMemcpyHostToDevice, p->s_h2d));
        CU(cudaEventRecord(e[1], p->s_h2d));
        CU(cudaStreamWaitEvent(p->s_comp, e[1], 0));
        if (k >= 2) CU(cudaStreamWaitEvent(p->s_comp, evs.slab(k - 2)[5], 0));
        CU(cudaEventRecord(e[2], p->s_comp));
        op(p, p->stage_in[b], ns, p->stage_out[b], p->s_comp);
        CU(cudaEventRecord(e[3], p->s_comp));
        CU(cudaStreamWaitEvent(p->s_d2h, e[3], 0));
        CU(cudaEventRecord(e[4], p->s_d2h));
        CU(cudaMemcpyAsync(hout + (size_t)s0 * out_per_slice, p->stage_out[b], (size_t)ns * out_per_slice * sizeof(float), cudaMemcpyDeviceToHost, p->s_d2h));
        CU(cudaEventRecord(e[5], p->s_d2h));
    }
    CU(cudaStreamSynchronize(p->s_d2h));
    CU(cudaStreamSynchronize(p->s_comp));
    auto t1 = std::chrono::steady_clock::now();
    tc_sched_stats &st = p->stats;
    st = tc_sched_stats{};
    TCS(evs.accumulate(nslab, st));
    st.wall_s = std::chrono::duration<double>(t1 - t0).count();
    st.n_slabs = nslab;
    st.h2d_bytes = (long long)S * in_per_slice * sizeof(float);
    st.d2h_bytes = (long long)S * out_per_slice * sizeof(float);
    st.overlap = overlap_fraction(st.h2d_s, st.compute_s, st.d2h_s, st.wall_s);
    return check_launch();
}

extern "C" tc_status tc_last_sched_stats(tc_plan *p, tc_sched_stats *out) {
    if (!p || !out) return fail(TC_EINVAL, "null argument");
    *out = p->stats;
    return TC_OK;
}

static tc_status run_op(tc_plan *p, slab_op op, const float *in, size_t in_per_slice, float *out, size_t out_per_slice, int S, void *stream) {
    if (!p || !in || !out) return fail(TC_EINVAL, "null argument");
    if (S <= 0) return fail(TC_EINVAL, "n_slices must be positive");
    const bool din = is_device_ptr(in), dout = is_device_ptr(out);
    if (din != dout) return fail(TC_EINVAL, "input and output must both be device or both be host pointers");
    int slab = 0;
    if (!din && p->max_slab == 0) {
        // host path: ~16 slabs so that the first copy in and the last copy out (not overlapped) are a small part, at most 64 slices per
        // slab by default (config 4, 128 slices: 8-slice slabs 86.8 ms per forward + adjoint, 32-slice slabs 98.8 ms)
        const int s = std::max(8, std::min(64, ((S + 15) / 16 + 7) / 8 * 8));
        TCS(ensure_scratch(p, S, &slab, s / 8));
        slab = std::min(slab, s);
    } else {
        TCS(ensure_scratch(p, S, &slab));
    }
    if (din) {
        cudaStream_t st = (cudaStream_t)stream;
        for (int s0 = 0; s0 < S; s0 += slab) {
            const int ns = std::min(slab, S - s0);
            op(p, in + (size_t)s0 * in_per_slice, ns, out + (size_t)s0 * out_per_slice, st);
        }
        return check_launch();
    }
    return run_streamed(p, op, in, in_per_slice, out, out_per_slice, S, slab);
}

extern "C" tc_status tc_radon(tc_plan *p, const float *volume, int n_slices, float *sinogram, void *stream) {
    if (!p) return fail(TC_EINVAL, "null plan");
    return run_op(p, forward_slab, volume, (size_t)p->d.n * p->d.n, sinogram, (size_t)p->d.na * p->d.nd, n_slices, stream);
}
extern "C" tc_status tc_backproject(tc_plan *p, const float *sinogram, int n_slices, float *volume, void *stream) {
    if (!p) return fail(TC_EINVAL, "null plan");
    p->fbp_filter = -1;
    return run_op(p, adjoint_slab, sinogram, (size_t)p->d.na * p->d.nd, volume, (size_t)p->d.n * p->d.n, n_slices, stream);
}

extern "C" tc_status tc_fbp(tc_plan *p, const float *sinogram, int n_slices, int filter, float *volume, void *stream) {
    if (!p) return fail(TC_EINVAL, "null plan");
    if (filter < TC_FILTER_RAMP || filter > TC_FILTER_BUTTERWORTH) return fail(TC_EINVAL, "unknown filter");
    p->fbp_filter = filter;                                   // launches read it while they are enqueued (below), not later
    const tc_status s = run_op(p, adjoint_slab, sinogram, (size_t)p->d.na * p->d.nd, volume, (size_t)p->d.n * p->d.n, n_slices, stream);
    p->fbp_filter = -1;
    return s;
}

extern "C" tc_status tc_radon1(const float *volume, int n_slices, int n, const float *angles, int n_angles, int n_det,
                               float center, float *sinogram) {
    tc_geom g{n, n_det, n_angles, angles, center, 2.0f, KB_W};
    tc_plan *p = nullptr;
    TCS(tc_plan_create(&g, 0, &p));
    tc_status s = tc_radon(p, volume, n_slices, sinogram, nullptr);
    if (s == TC_OK && cudaDeviceSynchronize() != cudaSuccess) s = fail(TC_ECUDA, "synchronize failed");
    tc_plan_destroy(p);
    return s;
}

// ---- Beer-Lambert pre-pass + projection -> sinogram reorder ----
extern "C" tc_status tc_preprocess(const float *proj, const float *flat, const float *dark, int n_angles, int n_slices, int n_det,
                                   float floor_, float *sinogram, void *stream) {
    if (!proj || !sinogram || n_angles <= 0 || n_slices <= 0 || n_det <= 0) return fail(TC_EINVAL, "bad argument");
    if (!(floor_ > 0.f)) return fail(TC_EINVAL, "floor must be positive (it bounds the argument of the logarithm)");
    const size_t n = (size_t)n_angles * n_slices * n_det, nf = (size_t)n_slices * n_det;
    const bool dev = is_device_ptr(proj);
    if (is_device_ptr(sinogram) != dev || (flat && is_device_ptr(flat) != dev) || (dark && is_device_ptr(dark) != dev))
        return fail(TC_EINVAL, "all arrays must be device pointers or all host pointers");
    cudaStream_t st = (cudaStream_t)stream;
    if (dev) { launch_preprocess(proj, flat, dark, n_angles, n_slices, n_det, floor_, sinogram, st); return check_launch(); }
    CallMem mem;
    float *dp = nullptr, *df = nullptr, *dd = nullptr, *ds = nullptr;
    CU(mem.alloc(&dp, n)); CU(mem.alloc(&ds, n));
    CU(cudaMemcpy(dp, proj, n * sizeof(float), cudaMemcpyHostToDevice));
    if (flat) { CU(mem.alloc(&df, nf)); CU(cudaMemcpy(df, flat, nf * sizeof(float), cudaMemcpyHostToDevice)); }
    if (dark) { CU(mem.alloc(&dd, nf)); CU(cudaMemcpy(dd, dark, nf * sizeof(float), cudaMemcpyHostToDevice)); }
    launch_preprocess(dp, df, dd, n_angles, n_slices, n_det, floor_, ds, nullptr);
    TCS(check_launch());
    CU(cudaMemcpy(sinogram, ds, n * sizeof(float), cudaMemcpyDeviceToHost));
    return TC_OK;
}

// ---- stage test hooks (unit tier): one complex plane through ONE stage, host arrays in natural order ----------
// F1 + F2: slices re / im (im nullable) -> the fine grid Ghat[k_y][k_x] of the plane re + i im (cells outside the sampled disc: 0)
extern "C" tc_status tc_stage_fine_grid(tc_plan *p, const float *re, const float *im, float *grid_out) {
    if (!p || !re || !grid_out) return fail(TC_EINVAL, "null argument");
    const DevPlan &d = p->d;
    const size_t nv = (size_t)d.n * d.n, ng2 = (size_t)d.G * d.G;
    int slab; TCS(ensure_scratch(p, 8, &slab));
    CallMem mem;
    float *vol = nullptr; float2 *nat = nullptr;
    CU(mem.alloc(&vol, 8 * nv)); CU(mem.alloc(&nat, ng2));
    CU(cudaMemset(vol, 0, 8 * nv * sizeof(float)));
    CU(cudaMemcpy(vol, re, nv * sizeof(float), cudaMemcpyHostToDevice));
    if (im) CU(cudaMemcpy(vol + nv, im, nv * sizeof(float), cudaMemcpyHostToDevice));
    CU(cudaMemset(p->grid, 0, ng2 * P * sizeof(float2)));
    launch_fwd_rows(d, vol, 8, 1, p->rowbuf, nullptr);
    launch_fwd_cols(d, p->rowbuf, 1, p->grid, nullptr);
    launch_grid_plane(p->grid, nat, d.G, 0, false, nullptr);
    TCS(check_launch());
    CU(cudaMemcpy(grid_out, nat, ng2 * sizeof(float2), cudaMemcpyDeviceToHost));
    return TC_OK;
}
// F3: fine grid Ghat[k_y][k_x] -> polar coefficients c[a][m mod nd] (before the centre phase; the Nyquist mode is not computed: 0)
extern "C" tc_status tc_stage_gather(tc_plan *p, const float *grid_in, float *cpol_out) {
    if (!p || !grid_in || !cpol_out) return fail(TC_EINVAL, "null argument");
    const DevPlan &d = p->d;
    const size_t ng2 = (size_t)d.G * d.G, ns = (size_t)d.na * d.nd;
    int slab; TCS(ensure_scratch(p, 8, &slab));
    CallMem mem;
    float2 *nat = nullptr, *natc = nullptr;
    CU(mem.alloc(&nat, ng2)); CU(mem.alloc(&natc, ns));
    CU(cudaMemcpy(nat, grid_in, ng2 * sizeof(float2), cudaMemcpyHostToDevice));
    CU(cudaMemset(p->grid, 0, ng2 * P * sizeof(float2)));
    CU(cudaMemset(p->cpol, 0, ns * P * sizeof(float2)));
    launch_grid_plane(p->grid, nat, d.G, 0, true, nullptr);
    launch_fwd_gather_tiles(d, p->grid, 1, p->cpol, nullptr);
    launch_cpol_plane(p->cpol, natc, ns, 0, false, nullptr);
    TCS(check_launch());
    CU(cudaMemcpy(cpol_out, natc, ns * sizeof(float2), cudaMemcpyDeviceToHost));
    return TC_OK;
}
// B2: polar coefficients c[a][m mod nd] -> fine grid Ghat[k_y][k_x] (cells outside the sampled disc: 0)
extern "C" tc_status tc_stage_spread(tc_plan *p, const float *cpol_in, float *grid_out) {
    if (!p || !cpol_in || !grid_out) return fail(TC_EINVAL, "null argument");
    const DevPlan &d = p->d;
    const size_t ng2 = (size_t)d.G * d.G, ns = (size_t)d.na * d.nd;
    int slab; TCS(ensure_scratch(p, 8, &slab));
    CallMem mem;
    float2 *nat = nullptr, *natc = nullptr;
    CU(mem.alloc(&nat, ng2)); CU(mem.alloc(&natc, ns));
    CU(cudaMemcpy(natc, cpol_in, ns * sizeof(float2), cudaMemcpyHostToDevice));
    CU(cudaMemset(p->grid, 0, ng2 * P * sizeof(float2)));
    CU(cudaMemset(p->cpol, 0, ns * P * sizeof(float2)));
    launch_cpol_plane(p->cpol, natc, ns, 0, true, nullptr);
    launch_adj_spread(d, p->cpol, 1, p->grid, nullptr);
    launch_grid_plane(p->grid, nat, d.G, 0, false, nullptr);
    TCS(check_launch());
    CU(cudaMemcpy(grid_out, nat, ng2 * sizeof(float2), cudaMemcpyDeviceToHost));
    return TC_OK;
}

// ---- prior test hook ---------------------------------------------------------------------------------
static tc_status check_prior(const tc_prior *pr) {
    if (!pr) return fail(TC_EINVAL, "null prior");
    if (!(pr->p >= 1.f && pr->p <= 2.f) || !(pr->sigma > 0.f) || !(pr->c > 0.f) || !(pr->lambda >= 0.f) || !(pr->L >= 0.f))
        return fail(TC_EINVAL, "prior: need 1 <= p <= 2, sigma > 0, c > 0, lambda >= 0, L >= 0");
    if (pr->neighbours != 0 && pr->neighbours != 26 && pr->neighbours != 10 && pr->neighbours != 6)
        return fail(TC_EINVAL, "prior: neighbours must be 26 (or 0 = 26), 10 or 6");
    return TC_OK;
}
static PriorDev prior_dev(const tc_prior *pr) {
    PriorDev pd{pr->p, pr->sigma, pr->c, pr->lambda, pr->nonneg != 0};
    pd.nbr = pr->neighbours == 0 ? 26 : pr->neighbours;
    return pd;
}

extern "C" tc_status tc_prior_eval(const float *volume, int S, int n, const tc_prior *pr, float *grad, double *value) {
    if (!volume || S <= 0 || n <= 0) return fail(TC_EINVAL, "bad argument");
    TCS(check_prior(pr));
    const size_t ne = (size_t)S * n * n;
    const bool dev = is_device_ptr(volume);
    if (grad && is_device_ptr(grad) != dev) return fail(TC_EINVAL, "volume and grad must both be device or both be host pointers");
    CallMem mem;
    float *dv = nullptr, *dg = nullptr; double *acc = nullptr;
    if (dev) dv = const_cast<float *>(volume);
    else { CU(mem.alloc(&dv, ne)); CU(cudaMemcpy(dv, volume, ne * sizeof(float), cudaMemcpyHostToDevice)); }
    if (grad) { if (dev) dg = grad; else CU(mem.alloc(&dg, ne)); }
    CU(mem.alloc(&acc, 16 + 4096));
    CU(cudaMemset(acc, 0, 16 * sizeof(double)));
    PriorDev pd = prior_dev(pr);
    pd.nonneg = 0;
    launch_prior(dv, pd, dg, value ? acc : nullptr, S, n, nullptr);
    TCS(check_launch());
    if (value) CU(cudaMemcpy(value, acc + 1, sizeof(double), cudaMemcpyDeviceToHost));
    if (grad && !dev) CU(cudaMemcpy(grad, dg, ne * sizeof(float), cudaMemcpyDeviceToHost));
    CU(cudaDeviceSynchronize());
    return TC_OK;
}

// ---- power iteration for the step constant (reading G15) ---------------------------------------------
extern "C" tc_status tc_power_iteration(tc_plan *p, int iters, double *lambda_hat) {
    if (!p || !lambda_hat || iters <= 0) return fail(TC_EINVAL, "bad argument");
    const DevPlan &d = p->d;
    const size_t nv = (size_t)d.n * d.n, nsn = (size_t)d.na * d.nd;
    int slab; TCS(ensure_scratch(p, 1, &slab));
    p->fbp_filter = -1;
    CallMem mem;
    float *v = nullptr, *w = nullptr, *s = nullptr;
    CU(mem.alloc(&v, nv)); CU(mem.alloc(&w, nv)); CU(mem.alloc(&s, nsn));
    std::vector<float> ones(nv, 1.0f);
    CU(cudaMemcpy(v, ones.data(), nv * sizeof(float), cudaMemcpyHostToDevice));
    double nv2 = (double)nv, lam = 0.0;
    for (int it = 0; it < iters; ++it) {
        forward_slab(p, v, 1, s, nullptr);
        adjoint_slab(p, s, 1, w, nullptr);
        CU(cudaMemsetAsync(p->acc, 0, 16 * sizeof(double), nullptr));
        launch_sumsq(w, nv, p->acc, 2, nullptr);
        double nw2;
        CU(cudaMemcpy(&nw2, p->acc + 2, sizeof(double), cudaMemcpyDeviceToHost));
        lam = std::sqrt(nw2 / nv2);
        launch_scale(w, (float)(1.0 / std::sqrt(nw2)), nv, nullptr);
        std::swap(v, w);
        nv2 = 1.0;
    }
    TCS(check_launch());
    CU(cudaDeviceSynchronize());
    *lambda_hat = lam;
    return TC_OK;
}

static tc_status mbir_streamed(tc_plan *p, const float *hb, int S, const tc_prior *pr, int iters, float *volume, tc_iter_log *log,
                               double L, int slab);      // tc_mbir_streamed.cuh

// ---- MBIR loop (M1-M5): monotone accelerated gradient with restart, reading G14 ----
// In core: x, x-, z, g and A x, A x-, A z, r, b live in device memory; A x is carried by linearity (one adjoint + one forward per
// iteration: A y = A x + beta (A x - A x-), A z = A y - alpha A g) and refreshed from scratch every AX_REFRESH iterations so that
// float32 rounding of the carried sinograms cannot accumulate over long runs.
// y is never stored: the update kernel forms it from x, x- while loading (M1 fused into M2/M3), and the residual kernel forms
// A y the same way.  A rejected candidate changes nothing but t (the next step has beta = 0, so x- is not even read).
constexpr int AX_REFRESH = 50;

// z-sharded form (comm != nullptr; P:L133 level-1 partition): this rank owns S consecutive slices of a taller volume.
// A and A^T are slice-wise, so only the prior couples the ranks: the volume arrays carry one halo slice towards each neighbour
// (lo / hi), the candidate's boundary slices are exchanged once per iteration (x and x- inherit their halos through the pointer
// rotation), and the terms of the objective are summed over ranks before the accept test, so every rank takes the same decision.
static tc_status mbir_in_core(tc_plan *p, const float *sinogram, int S, const tc_prior *pr, int iters, float *volume, tc_iter_log *log,
                              double L, cudaStream_t st, bool dev_b, bool dev_v, bool *retry_streamed, const tc_comm *comm = nullptr) {
    const DevPlan &d = p->d;
    const size_t vps = (size_t)d.n * d.n, sps = (size_t)d.na * d.nd;
    const int lo = comm && comm->send_down ? 1 : 0, hi = comm && comm->send_up ? 1 : 0, Sx = S + lo + hi;
    const size_t nv = (size_t)S * vps, ns = (size_t)S * sps, nvx = (size_t)Sx * vps;
    *retry_streamed = false;
    int slab; TCS(ensure_scratch(p, S, &slab, 16));           // at most 16 groups of FFT scratch: the state below needs the memory
    if (!p->s_aux) {
        CU(cudaStreamCreateWithFlags(&p->s_aux, cudaStreamNonBlocking));
        for (auto &ev : p->ev_aux) CU(cudaEventCreateWithFlags(&ev, cudaEventDisableTiming));
    }
    CallMem mem;
    float *vb[4] = {nullptr}, *sb[5] = {nullptr};
    bool ok = true;
    for (int i = 0; i < 4 && ok; ++i) ok = mem.alloc(&vb[i], nvx) == cudaSuccess;
    for (int i = 0; i < 5 && ok; ++i) {
        if (i == 4 && dev_b) { sb[4] = const_cast<float *>(sinogram); continue; }
        ok = mem.alloc(&sb[i], ns) == cudaSuccess;
    }
    if (!ok) {
        *retry_streamed = !dev_b && !dev_v;
        return fail(TC_ENOMEM, "tc_mbir: the in-core working set (4 volumes + 5 sinograms) does not fit in device memory; "
                               "pass host pointers to stream the problem");
    }
    // xe, xme, ze, ge: arrays of Sx slices (halo, core, halo); x, xm, z, gv: their core parts
    float *xe = vb[0], *xme = vb[1], *ze = vb[2], *ge = vb[3];
    const size_t co = (size_t)lo * vps;
    float *x = xe + co, *xm = xme + co, *z = ze + co, *gv = ge + co;
    float *Ax = sb[0], *Axm = sb[1], *Az = sb[2], *r = sb[3], *b = sb[4];
    if (!dev_b) CU(cudaMemcpyAsync(b, sinogram, ns * sizeof(float), cudaMemcpyHostToDevice, st));
    CU(cudaMemsetAsync(xe, 0, nvx * sizeof(float), st)); CU(cudaMemsetAsync(xme, 0, nvx * sizeof(float), st));
    CU(cudaMemsetAsync(ze, 0, nvx * sizeof(float), st));
    CU(cudaMemsetAsync(Ax, 0, ns * sizeof(float), st)); CU(cudaMemsetAsync(Axm, 0, ns * sizeof(float), st));
    CU(cudaMemsetAsync(p->acc, 0, 16 * sizeof(double), st));
    launch_sumsq(b, ns, p->acc, 2, st);
    double h[8];
    CU(cudaMemcpyAsync(h, p->acc, 8 * sizeof(double), cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
    TCS(check_launch());
    if (comm && comm->allreduce(comm->ctx, h + 2, 1) != 0) return fail(TC_ECUDA, "tc_mbir_sharded: allreduce callback failed");
    double Fx = 0.5 * h[2], t = 1.0;
    const PriorDev pd = prior_dev(pr);
    const float invL = (float)(1.0 / L);
    p->fbp_filter = -1;
    auto slabbed = [&](slab_op op, const float *in, size_t ips, float *out, size_t ops) {
        for (int s0 = 0; s0 < S; s0 += slab) op(p, in + (size_t)s0 * ips, std::min(slab, S - s0), out + (size_t)s0 * ops, st);
    };
    bool r_ready = false;                                                 // r holds the coming iteration's residual (written by k_candidate_sino)
    auto t_iter = std::chrono::steady_clock::now();                       // tc_iter_log.ms: from one accept test's synchronisation to the next
    for (int it = 0; it < iters; ++it) {
        NvtxRange nv_it("tc_mbir iteration");
        const double tp = 0.5 * (1.0 + std::sqrt(1.0 + 4.0 * t * t));
        const float beta = (float)((t - 1.0) / tp);
        if (it > 0 && it % AX_REFRESH == 0) {                             // A x, A x- from scratch
            slabbed(forward_slab, x, vps, Ax, sps);
            slabbed(forward_slab, xm, vps, Axm, sps);
        }
        if (it > 0 && it % AX_REFRESH == 0) r_ready = false;
        if (!r_ready) launch_residual(Ax, Axm, b, beta, r, ns, st);       // M1 (sinogram part): r = A y - b (else: left there by the last candidate kernel)
        slabbed(adjoint_slab, r, sps, gv, vps);                           // A^T (A y - b)
        CU(cudaMemsetAsync(p->acc, 0, 16 * sizeof(double), st));
        float alpha = invL;
        if (pr->mm_step) {
            // majorise-minimise step length along -g (G23): alpha = <g, g> / (||A g||^2 + lambda c(y; g)),
            // c = sum over pairs of w h'(D)/D (g_m - g_n)^2, D = y_m - y_n: needs g and A g before z
            launch_update(x, xm, beta, gv, pd, 0.f, gv, nullptr, S, d.n, st);                 // g = A^T r + lambda grad H(y)
            slabbed(forward_slab, gv, vps, r, sps);                                          // A g
            launch_sumsq(gv, nv, p->acc, 4, st);
            launch_sumsq(r, ns, p->acc, 5, st);
            launch_prior_curvature(x, xm, beta, gv, pd, p->acc, 6, S, d.n, st);
            CU(cudaMemcpyAsync(h, p->acc, 8 * sizeof(double), cudaMemcpyDeviceToHost, st));
            CU(cudaStreamSynchronize(st));
            const double den = h[5] + (double)pr->lambda * h[6];
            alpha = den > 0.0 ? (float)(h[4] / den) : invL;
            launch_step(x, xm, beta, gv, alpha, pd.nonneg, z, nv, st);                        // z = y - alpha g (projected if nonneg)
        } else {
            launch_update(xe, xme, beta, ge, pd, invL, ge, ze, Sx, d.n, st, lo, S);           // M2 + M3: g, z = y - g / L on the core
        }
        // M4.  The data term streams five sinograms (HBM-bound), the prior term is a stencil (MUFU / issue-bound): unless ranks have to
        // exchange halos in between, the first runs on a second stream beside the second.
        cudaStream_t sd = st;
        if (!comm && p->s_aux) sd = p->s_aux;
        if (pd.nonneg) {                                                  // projected candidate: z is not linear in g, so A z itself
            slabbed(forward_slab, z, vps, r, sps);
            if (sd != st) { CU(cudaEventRecord(p->ev_aux[0], st)); CU(cudaStreamWaitEvent(sd, p->ev_aux[0], 0)); }
            launch_candidate_sino(r, nullptr, nullptr, b, 0.f, 0.f, Az, p->acc, ns, sd);      // M4: Az = A z
        } else {
            if (!pr->mm_step) slabbed(forward_slab, gv, vps, r, sps);     // A g
            if (sd != st) { CU(cudaEventRecord(p->ev_aux[0], st)); CU(cudaStreamWaitEvent(sd, p->ev_aux[0], 0)); }
            // M4: Az = A y - alpha A g; the same pass leaves, in place of A g, the residual of the next iteration for the case that this
            // candidate is accepted without a restart (the momentum of that iteration is known now: t becomes tp)
            const double tp2 = 0.5 * (1.0 + std::sqrt(1.0 + 4.0 * tp * tp));
            launch_candidate_sino(Ax, Axm, r, b, beta, alpha, Az, p->acc, ns, sd, r, (float)((tp - 1.0) / tp2));
        }
        if (sd != st) CU(cudaEventRecord(p->ev_aux[1], sd));
        if (comm) {                                                       // the candidate's boundary slices go to the neighbours' halos
            if (lo) CU(cudaMemcpyAsync(comm->send_down, z, vps * sizeof(float), cudaMemcpyDeviceToDevice, st));
            if (hi) CU(cudaMemcpyAsync(comm->send_up, z + (size_t)(S - 1) * vps, vps * sizeof(float), cudaMemcpyDeviceToDevice, st));
            CU(cudaStreamSynchronize(st));
            if (comm->exchange(comm->ctx) != 0) return fail(TC_ECUDA, "tc_mbir_sharded: halo exchange callback failed");
            if (lo) CU(cudaMemcpyAsync(ze, comm->recv_down, vps * sizeof(float), cudaMemcpyDeviceToDevice, st));
            if (hi) CU(cudaMemcpyAsync(ze + (size_t)(Sx - 1) * vps, comm->recv_up, vps * sizeof(float), cudaMemcpyDeviceToDevice, st));
        }
        launch_prior(z, pd, nullptr, p->acc, S + hi, d.n, st, S);         // pairs are owned by their lower slice: the core's, up to the upper halo
        if (sd != st) CU(cudaStreamWaitEvent(st, p->ev_aux[1], 0));
        if (pr->grad_restart) launch_dot_gzx(gv, z, x, nv, p->acc, 3, st);
        CU(cudaMemcpyAsync(h, p->acc, 4 * sizeof(double), cudaMemcpyDeviceToHost, st));
        CU(cudaStreamSynchronize(st));
        TCS(check_launch());
        if (comm && comm->allreduce(comm->ctx, h, 4) != 0) return fail(TC_ECUDA, "tc_mbir_sharded: allreduce callback failed");
        const double Fz = h[0] + (double)pr->lambda * h[1];
        const double margin = (Fx - Fz) / Fx;
        const bool accept = Fz <= Fx;                                     // M5
        const bool restarted = pr->grad_restart && accept && h[3] > 0.0;
        if (accept) {
            float *oe = xme; xme = xe; xe = ze; ze = oe;
            x = xe + co; xm = xme + co; z = ze + co;
            float *oa = Axm; Axm = Ax; Ax = Az; Az = oa;
            Fx = Fz; t = restarted ? 1.0 : tp;
            r_ready = !restarted && !pd.nonneg;                           // r already holds A y - b of the next iteration
        } else {
            r_ready = false;
            t = 1.0;                                                      // restart: the next step is a plain gradient step from x (beta = 0)
        }
        if (log) { log[it].F = Fx; log[it].data = h[0]; log[it].prior = h[1]; log[it].margin = margin; log[it].beta = beta; log[it].accepted = accept ? 1 : 0;
                   log[it].dot = pr->grad_restart ? h[3] : 0.0; log[it].restarted = restarted ? 1 : 0; log[it].alpha = alpha;
                   const auto t_now = std::chrono::steady_clock::now(); log[it].ms = (float)std::chrono::duration<double, std::milli>(t_now - t_iter).count(); t_iter = t_now; }
    }
    CU(cudaMemcpyAsync(volume, x, nv * sizeof(float), dev_v ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
    p->stats = tc_sched_stats{};
    return check_launch();
}

extern "C" tc_status tc_mbir(tc_plan *p, const float *sinogram, int S, const tc_prior *pr, int iters, float *volume,
                             tc_iter_log *log, void *stream) {
    if (!p || !sinogram || !volume) return fail(TC_EINVAL, "null argument");
    if (S <= 0 || iters < 0) return fail(TC_EINVAL, "n_slices must be positive, iters non-negative");
    TCS(check_prior(pr));
    const DevPlan &d = p->d;
    const size_t nv = (size_t)S * d.n * d.n, ns = (size_t)S * d.na * d.nd;
    double L = pr->L;
    if (L <= 0) {
        double lam_hat; TCS(tc_power_iteration(p, 10, &lam_hat));
        L = 1.05 * lam_hat + (double)pr->lambda * 4.0 / ((double)pr->c * pr->sigma * pr->sigma);
    }
    const bool dev_b = is_device_ptr(sinogram), dev_v = is_device_ptr(volume);
    const bool host = !dev_b && !dev_v;
    auto stream_it = [&]() -> tc_status {
        if (pr->mm_step) return fail(TC_EUNSUPPORTED, "tc_mbir: mm_step is available in core only");
        const bool forced = p->max_slab > 0 && p->max_slab < S;
        int slab_s = forced ? p->max_slab : 32, have = 0;
        TCS(ensure_scratch(p, slab_s + 1, &have, (slab_s + 1 + 7) / 8));   // scratch for the core and the slice above it
        if (have < slab_s + 1) slab_s = std::max(1, have - 1);
        return mbir_streamed(p, sinogram, S, pr, iters, volume, log, L, slab_s);
    };
    if (host) {
        // host-resident problem: stream it when the caller caps the slab (max_slab_slices) or when the in-core working set
        // (4 volumes + 5 sinograms + at most 16 groups of FFT scratch, the same bound mbir_in_core uses) does not fit
        size_t fr = 0, tot = 0;
        CU(cudaMemGetInfo(&fr, &tot));
        const double have = (double)fr + (double)p->ng_alloc * group_bytes(p);
        const double need = 4.0 * nv * 4 + 5.0 * ns * 4 + (double)group_bytes(p) * std::min((S + 7) / 8, 16);
        if ((p->max_slab > 0 && p->max_slab < S) || need > 0.9 * have) return stream_it();
    }
    bool retry = false;
    const tc_status s = mbir_in_core(p, sinogram, S, pr, iters, volume, log, L, (cudaStream_t)stream, dev_b, dev_v, &retry);
    if (s == TC_ENOMEM && retry) return stream_it();                      // the estimate was wrong (fragmentation, other tenants): stream instead
    return s;
}

// ---- z-sharded MBIR: one rank of a volume partitioned along the rotation axis ----
extern "C" tc_status tc_mbir_sharded(tc_plan *p, const float *sinogram, int S, const tc_prior *pr, int iters, float *volume,
                                     tc_iter_log *log, const tc_comm *comm, void *stream) {
    if (!p || !sinogram || !volume || !comm) return fail(TC_EINVAL, "null argument");
    if (S <= 0 || iters < 0) return fail(TC_EINVAL, "n_slices must be positive, iters non-negative");
    if (!comm->exchange || !comm->allreduce) return fail(TC_EINVAL, "tc_comm: exchange and allreduce callbacks are required");
    if ((comm->send_down == nullptr) != (comm->recv_down == nullptr) || (comm->send_up == nullptr) != (comm->recv_up == nullptr))
        return fail(TC_EINVAL, "tc_comm: send / recv buffers must come in pairs");
    TCS(check_prior(pr));
    if (pr->mm_step) return fail(TC_EUNSUPPORTED, "tc_mbir_sharded: mm_step is not available");
    if (!(pr->L > 0.f)) return fail(TC_EINVAL, "tc_mbir_sharded: pass the step constant L (the same on every rank)");
    if (!is_device_ptr(sinogram) || !is_device_ptr(volume)) return fail(TC_EINVAL, "tc_mbir_sharded: device pointers only");
    for (const float *q : {comm->send_down, comm->recv_down, comm->send_up, comm->recv_up})
        if (q && !is_device_ptr(q)) return fail(TC_EINVAL, "tc_comm: halo buffers must be device memory");
    bool retry = false;
    return mbir_in_core(p, sinogram, S, pr, iters, volume, log, (double)pr->L, (cudaStream_t)stream, true, true, &retry, comm);
}
