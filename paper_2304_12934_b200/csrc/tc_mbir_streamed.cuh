// Included by tc_api.cu: out-of-core MBIR (S1 + M1-M5).  Volume and sinogram live in host memory (Fig. 3);
// every iteration streams z-slabs through the device on three streams (H2D, compute, D2H), two buffer sets.
//
// The link to the host is the bottleneck here, so unlike the in-core loop (which carries A x by linearity) this one
// RECOMPUTES A y every iteration (two forwards + one adjoint; equal up to rounding): no sinogram-sized state
// crosses PCIe except b.  Per slab with core slices [s0, s1) the device needs
//   x, x-  on [s0 - 1, s1 + 2)   (y there feeds the neighbourhood gradient on [s0, s1 + 1))
//   b      on [s0, s1 + 1)       (z on the slice above the core is needed by the prior pairs the core owns)
// and returns z on the core.  Slab edges inside the volume are not boundaries (reading G12): the halo is real data.
//
// Host-resident state is TWO volumes, not three: U holds x, V holds x- and is overwritten IN PLACE by the candidate z, slab by
// slab, as it comes back.  That is safe because (a) x- is dead after the iteration whatever the decision (accept: x- <- x;
// reject: t <- 1, so the next step has beta = 0 and never reads x-), and (b) the one slice of x- that slab k + 1 still needs
// after slab k's z has landed on it (its lower halo, slice s1 - 1) is taken from slab k's device buffer instead of the host.
// One of the two volumes is the caller's output array (page-locked for the call if it is pageable); the other one is pinned
// by the library.  Accept swaps the roles of U and V (pointers only).  A volume that is still all zero (x before the first
// accepted step, x- before the second) is never read from the host: its slabs are cleared on the device.

struct MbirSlabBufs {
    float *x = nullptr, *xm = nullptr, *b = nullptr;   // inputs
    float *z = nullptr;                                // output (computed on the op range, the core goes back)
};
struct HostVol { float *p = nullptr; bool zero = true; };   // zero: never written; stands for an all-zero volume

static tc_status mbir_streamed(tc_plan *p, const float *hb, int S, const tc_prior *pr, int iters, float *volume, tc_iter_log *log,
                               double L, int slab) {
    const DevPlan &d = p->d;
    const size_t vps = (size_t)d.n * d.n, sps = (size_t)d.na * d.nd;
    const size_t nv = (size_t)S * vps, ns = (size_t)S * sps;
    const float invL = (float)(1.0 / L);
    const PriorDev pd = prior_dev(pr);
    const size_t F4 = sizeof(float);
    TCS(ensure_streams(p));
    p->fbp_filter = -1;
    auto t_setup = std::chrono::steady_clock::now();
    CallMem mem;
    // ---- host state: the caller's volume + one pinned volume ----
    HostVol U, V;
    if (mem.pin(volume, nv * F4)) U.p = volume;
    else if (mem.alloc_host(&U.p, nv) != cudaSuccess) return fail(TC_ENOMEM, "tc_mbir (streamed): pinned host volume");
    if (mem.alloc_host(&V.p, nv) != cudaSuccess) return fail(TC_ENOMEM, "tc_mbir (streamed): pinned host volume");
    mem.pin(hb, ns * F4);                                     // pageable sinogram: locked for the call, else its copies would not overlap
    // ---- device buffers ----
    const int ext_v = slab + 3, ext_s = slab + 1;            // slices of the volume-side and sinogram-side slab arrays
    MbirSlabBufs B[2];
    float *y = nullptr, *gv = nullptr, *Ay = nullptr, *r = nullptr;
    bool ok = true;
    for (int k = 0; k < 2 && ok; ++k)
        ok = mem.alloc(&B[k].x, ext_v * vps) == cudaSuccess && mem.alloc(&B[k].xm, ext_v * vps) == cudaSuccess &&
             mem.alloc(&B[k].z, ext_v * vps) == cudaSuccess && mem.alloc(&B[k].b, ext_s * sps) == cudaSuccess;
    ok = ok && mem.alloc(&y, ext_v * vps) == cudaSuccess && mem.alloc(&gv, ext_v * vps) == cudaSuccess &&
         mem.alloc(&Ay, ext_s * sps) == cudaSuccess && mem.alloc(&r, ext_s * sps) == cudaSuccess;
    if (!ok) return fail(TC_ENOMEM, "tc_mbir (streamed): device slab buffers");
    const int nslab = (S + slab - 1) / slab;
    SlabEvents evs;
    CU(evs.create((size_t)nslab * 6));
    cudaStream_t sh = p->s_h2d, sc = p->s_comp, sd = p->s_d2h;
    tc_sched_stats &stt = p->stats;
    stt = tc_sched_stats{};

    // F(x = 0) = 1/2 ||b||^2, slab by slab
    CU(cudaMemsetAsync(p->acc, 0, 16 * sizeof(double), sc));
    for (int k = 0; k < nslab; ++k) {
        const int s0 = k * slab, nsl = std::min(slab, S - s0);
        CU(cudaMemcpyAsync(B[0].b, hb + (size_t)s0 * sps, (size_t)nsl * sps * F4, cudaMemcpyHostToDevice, sc));
        launch_sumsq(B[0].b, (size_t)nsl * sps, p->acc, 2, sc);
    }
    double h[4];
    CU(cudaMemcpyAsync(h, p->acc, 3 * sizeof(double), cudaMemcpyDeviceToHost, sc));
    CU(cudaStreamSynchronize(sc));
    TCS(check_launch());
    double Fx = 0.5 * h[2], t = 1.0;
    auto t_begin = std::chrono::steady_clock::now();
    stt.setup_s = std::chrono::duration<double>(t_begin - t_setup).count();
    auto t_iter = std::chrono::steady_clock::now();
    for (int it = 0; it < iters; ++it) {
        const double tp = 0.5 * (1.0 + std::sqrt(1.0 + 4.0 * t * t));
        const float beta = (float)((t - 1.0) / tp);
        const bool need_xm = beta != 0.f;                     // beta = 0 (first step, step after a restart): y = x, x- is not read
        CU(cudaMemsetAsync(p->acc, 0, 16 * sizeof(double), sc));
        for (int k = 0; k < nslab; ++k) {
            MbirSlabBufs &b = B[k & 1];
            cudaEvent_t *ek = evs.slab(k);
            const int s0 = k * slab, s1 = std::min(S, s0 + slab);
            const int a0 = std::max(0, s0 - 1), a1 = std::min(S, s1 + 2), e1 = std::min(S, s1 + 1);
            const int nva = a1 - a0, nop = e1 - s0, ncore = s1 - s0, off = s0 - a0;
            // H2D (the buffers of slab k - 2 are free once its compute is done)
            if (k >= 2) CU(cudaStreamWaitEvent(sh, evs.slab(k - 2)[3], 0));
            CU(cudaEventRecord(ek[0], sh));
            if (U.zero) CU(cudaMemsetAsync(b.x, 0, (size_t)nva * vps * F4, sh));
            else { CU(cudaMemcpyAsync(b.x, U.p + (size_t)a0 * vps, (size_t)nva * vps * F4, cudaMemcpyHostToDevice, sh)); stt.h2d_bytes += (long long)((size_t)nva * vps * F4); }
            if (need_xm) {
                if (V.zero) CU(cudaMemsetAsync(b.xm, 0, (size_t)nva * vps * F4, sh));
                else {
                    // the lower halo slice (s0 - 1) has already been overwritten on the host by slab k - 1's z: take it from that slab's device copy
                    if (off == 1) {
                        const MbirSlabBufs &pb = B[(k - 1) & 1];
                        const int pa0 = std::max(0, (k - 1) * slab - 1);
                        CU(cudaMemcpyAsync(b.xm, pb.xm + (size_t)(a0 - pa0) * vps, vps * F4, cudaMemcpyDeviceToDevice, sh));
                    }
                    CU(cudaMemcpyAsync(b.xm + (size_t)off * vps, V.p + (size_t)s0 * vps, (size_t)(nva - off) * vps * F4, cudaMemcpyHostToDevice, sh));
                    stt.h2d_bytes += (long long)((size_t)(nva - off) * vps * F4);
                }
            }
            CU(cudaMemcpyAsync(b.b, hb + (size_t)s0 * sps, (size_t)nop * sps * F4, cudaMemcpyHostToDevice, sh));
            stt.h2d_bytes += (long long)((size_t)nop * sps * F4);
            CU(cudaEventRecord(ek[1], sh));
            // compute
            CU(cudaStreamWaitEvent(sc, ek[1], 0));
            if (k >= 2) CU(cudaStreamWaitEvent(sc, evs.slab(k - 2)[5], 0));
            CU(cudaEventRecord(ek[2], sc));
            const float *yv = b.x;
            if (need_xm) { launch_extrapolate(b.x, b.xm, beta, y, (size_t)nva * vps, sc); yv = y; }   // M1
            forward_slab(p, yv + (size_t)off * vps, nop, Ay, sc);                                  // A y on the core and one slice above
            launch_residual(Ay, Ay, b.b, 0.f, r, (size_t)nop * sps, sc);                           // r = A y - b
            adjoint_slab(p, r, nop, gv + (size_t)off * vps, sc);                                   // A^T (A y - b) on the core and one slice above
            launch_update(yv, nullptr, 0.f, gv, pd, invL, gv, b.z, nva, d.n, sc, off, nop);       // M2 + M3
            if (pd.nonneg) {                                                                       // projected candidate: A z itself
                forward_slab(p, b.z + (size_t)off * vps, ncore, r, sc);
                launch_candidate_sino(r, nullptr, nullptr, b.b, 0.f, 0.f, r, p->acc, (size_t)ncore * sps, sc);      // M4 (A z is not kept)
            } else {
                forward_slab(p, gv + (size_t)off * vps, ncore, r, sc);                             // A g on the core
                launch_candidate_sino(Ay, nullptr, r, b.b, 0.f, invL, r, p->acc, (size_t)ncore * sps, sc);          // M4 (A z is not kept)
            }
            launch_prior(b.z + (size_t)off * vps, pd, nullptr, p->acc, nop, d.n, sc, ncore);
            if (pr->grad_restart) launch_dot_gzx(gv + (size_t)off * vps, b.z + (size_t)off * vps, b.x + (size_t)off * vps, (size_t)ncore * vps, p->acc, 3, sc);
            CU(cudaEventRecord(ek[3], sc));
            // D2H: z lands on x- (in place, see the header); slab k + 1's H2D of x- starts at its own core, beyond this range
            CU(cudaStreamWaitEvent(sd, ek[3], 0));
            if (need_xm && !V.zero) CU(cudaStreamWaitEvent(sd, ek[1], 0));                         // (implied by ek[3]; kept explicit: V[s0, s1) was read by this slab's H2D)
            CU(cudaEventRecord(ek[4], sd));
            CU(cudaMemcpyAsync(V.p + (size_t)s0 * vps, b.z + (size_t)off * vps, (size_t)ncore * vps * F4, cudaMemcpyDeviceToHost, sd));
            CU(cudaEventRecord(ek[5], sd));
            stt.d2h_bytes += (long long)((size_t)ncore * vps * F4);
        }
        CU(cudaMemcpyAsync(h, p->acc, 4 * sizeof(double), cudaMemcpyDeviceToHost, sc));
        CU(cudaStreamSynchronize(sc));
        CU(cudaStreamSynchronize(sd));
        CU(cudaStreamSynchronize(sh));
        TCS(check_launch());
        TCS(evs.accumulate(nslab, stt));
        V.zero = false;                                                                            // V now holds the candidate z
        const double Fz = h[0] + (double)pr->lambda * h[1];
        const double margin = (Fx - Fz) / Fx;
        const bool accept = Fz <= Fx;                                                             // M5
        const bool restarted = pr->grad_restart && accept && h[3] > 0.0;
        if (accept) { std::swap(U, V); Fx = Fz; t = restarted ? 1.0 : tp; }                       // x <- z, x- <- x: the two volumes swap roles
        else t = 1.0;                                                                              // V holds a dead candidate; the next step (beta = 0) does not read it
        if (log) { log[it].F = Fx; log[it].data = h[0]; log[it].prior = h[1]; log[it].margin = margin; log[it].beta = beta; log[it].accepted = accept ? 1 : 0;
                   log[it].dot = pr->grad_restart ? h[3] : 0.0; log[it].restarted = restarted ? 1 : 0; log[it].alpha = invL;
                   const auto t_now = std::chrono::steady_clock::now(); log[it].ms = (float)std::chrono::duration<double, std::milli>(t_now - t_iter).count(); t_iter = t_now; }
    }
    auto t_end = std::chrono::steady_clock::now();
    stt.wall_s = std::chrono::duration<double>(t_end - t_begin).count();                          // the iterations
    // hand-over: x is in U; nothing to do if that is the caller's array
    if (U.zero) memset(volume, 0, nv * F4);
    else if (U.p != volume) memcpy(volume, U.p, nv * F4);
    stt.handover_s = std::chrono::duration<double>(std::chrono::steady_clock::now() - t_end).count();
    stt.n_slabs = nslab;
    stt.overlap = overlap_fraction(stt.h2d_s, stt.compute_s, stt.d2h_s, stt.wall_s);
    return check_launch();
}
