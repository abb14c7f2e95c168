// plan_run.inl -- the iteration drivers of PlanImpl<T> (included after plan_impl.inl).
//
// Nothing in the loops below waits for the device: the step length, the Armijo decision, the
// stopping rules and the traces are computed by device code (sgp_dev.cuh); kernels return at once when
// the device status is no longer "running".  The host reads the control block only every
// `check_every` iterations (once, at the end, for a fixed iteration count).
namespace sgpk {

template <typename T>
int PlanImpl<T>::ensure_trace(int max_iter, const sgp_result *res, Trace *tr, cudaStream_t st)
{
    const int need = max_iter + 1;
    if (need > trace_cap) {
        free_trace();
        const size_t cap = ((size_t)need + 1) & ~(size_t)1;     // even: the int arrays stay 8-byte aligned
        SGP_CUDA_TRY(cudaMalloc((void **)&trJ, (5 * sizeof(double) + 2 * sizeof(int)) * cap));      // one block
        trA = trJ + cap; trL = trA + cap; fA = trL + cap; fL = fA + cap;
        trR = reinterpret_cast<int *>(fL + cap); trB = trR + cap;
        trace_cap = (int)cap;
    }
    SGP_CUDA_TRY(cudaMemsetAsync(trJ, 0, (5 * sizeof(double) + 2 * sizeof(int)) * (size_t)trace_cap, st));
    tr->J = trJ; tr->alpha = trA; tr->lambda = trL; tr->rule = trR; tr->backtracks = trB;
    tr->force_alpha = nullptr; tr->force_lambda = nullptr;
    if (res->force_alpha && max_iter > 0) {
        SGP_CUDA_TRY(cudaMemcpyAsync(fA, res->force_alpha, sizeof(double) * max_iter, cudaMemcpyHostToDevice, st));
        tr->force_alpha = fA;
    }
    if (res->force_lambda && max_iter > 0) {
        SGP_CUDA_TRY(cudaMemcpyAsync(fL, res->force_lambda, sizeof(double) * max_iter, cudaMemcpyHostToDevice, st));
        tr->force_lambda = fL;
    }
    return SGP_OK;
}

// One SGP iteration: K2 column pass with conj(K^) summed over the images, K3 inverse rows + lazy
// f update + gradient + BB sums + step length, K4 projection + row FFT of d, K5 column pass with K^_j, K6 inverse rows +
// u_j + J(lambda = 1) + Armijo test + book-keeping (fused form: also q(k+1), the ratio and its row FFT), then the tail
// K7 backtracks (elementwise; returns at once when lambda = 1 was accepted) and K1 = ratio + row FFT of iteration k + 1.
// The ratio kernel of the FIRST iteration is enqueued by run() before the loop.
//
// Experiment (opt.use_graph bit 5, off by default): inside a captured graph the tail becomes a fork -- K1 in its
// "lambda = 1 accepted" instance BESIDE K7 -> K1 in its repair instance, the next K2 joining both -- which takes the two
// kernels that usually return at once off the critical path.  Measured: the fork / join edges cost more than the
// 2.7 us they hide (C4c 7660 vs 8110 it/s, C0 14.6 vs 17.3 kit/s), so the tail stays in stream order.
template <typename T>
int PlanImpl<T>::enqueue_ratio(const RowParams<T> &Pb, int lazy, cudaStream_t st)
{
    cur_slot = SGP_PROF_K1;
    RowParams<T> P = Pb; P.lazy = lazy; P.in0 = Gp; P.in1 = q; P.in2 = Bp; P.in3 = u; P.out0 = q;
    int rc = launch_row(k_rowf[RF_RATIO], P, p, st);
    cur_slot = -1;
    return rc;
}

template <typename T>
int PlanImpl<T>::enqueue_backtrack(const DevOpts &o, const Trace &tr, const double *bconst, int b_is_array, cudaStream_t st)
{
    cur_slot = SGP_PROF_K7;
    {
        BtParams<T> U;
        memset(&U, 0, sizeof(U));
        U.G = G; U.o = o; U.tr = tr; U.ct = ct; U.q = q; U.u = u; U.g = Gp; U.b = Bp;
        U.plane = n; U.qbuf = n * (size_t)p; U.b_is_array = b_is_array; U.part = part_bt;
        for (int j = 0; j < p; ++j) U.bconst[j] = bconst[j];
        ProfScope ps(this, st);
        backtrack_kernel<T><<<bt_grid, 256, 0, st>>>(U);
        launches++;
        SGP_CUDA_TRY(cudaGetLastError());
    }
    cur_slot = -1;
    return SGP_OK;
}

template <typename T>
int PlanImpl<T>::enqueue_sgp_iteration(const RowParams<T> &Pb, const DevOpts &o, const Trace &tr, const double *bconst,
                                       int b_is_array, cudaStream_t st)
{
    int rc;
    cur_slot = SGP_PROF_K2;
    {   // K2 (a2)
        ColParams<T> Q = col_params(); Q.check_status = 1;
        if ((rc = launch_col(k_conj_run, Q, st))) return rc;
    }
    cur_slot = SGP_PROF_K3;
    {   // K3 (a10 for f, a3, a5, a6)
        RowParams<T> P = Pb; P.lazy = 1; P.in0 = f; P.in1 = d; P.out0 = grad; P.out1 = f; P.part = part_bb;
        if ((rc = launch_row(k_rowi[RI_GRAD], P, 1, st))) return rc;
    }
    cur_slot = SGP_PROF_K4;
    {   // K4 (a4, a7)
        RowParams<T> P = Pb; P.in0 = f; P.in1 = grad; P.out0 = d; P.part = part_gd;
        if ((rc = launch_row(k_rowf[RF_PROJECT], P, 1, st))) return rc;
    }
    cur_slot = SGP_PROF_K5;
    {   // K5 (a8)
        ColParams<T> Q = col_params(); Q.check_status = 1;
        if ((rc = launch_col(k_mult_run, Q, st))) return rc;
    }
    cur_slot = SGP_PROF_K6;
    {   // K6 (a8 tail, a9 at lambda = 1, a11)
        RowParams<T> P = Pb; P.in0 = Gp; P.in1 = q; P.in2 = Bp; P.out0 = u; P.part = part_J; P.part2 = part_gd;
        if ((rc = launch_row(k_rowi[fuse_ls ? RI_LSF : RI_LS], P, p, st))) return rc;
    }
    cur_slot = -1;
    // ---- tail: K7 (a9 backtracks, a11) and K1 of the next iteration (a10 for q, a1)
    if (st == cap_stream && cap_stream2 && (opt.use_graph & 32)) {
        SGP_CUDA_TRY(cudaEventRecord(ev_fork, st));
        SGP_CUDA_TRY(cudaStreamWaitEvent(cap_stream2, ev_fork, 0));
        if ((rc = enqueue_backtrack(o, tr, bconst, b_is_array, cap_stream2))) return rc;
        if ((rc = enqueue_ratio(Pb, 2, cap_stream2))) return rc;
        SGP_CUDA_TRY(cudaEventRecord(ev_join, cap_stream2));
        if ((rc = enqueue_ratio(Pb, 1, st))) return rc;
        SGP_CUDA_TRY(cudaStreamWaitEvent(st, ev_join, 0));
    } else {
        if ((rc = enqueue_backtrack(o, tr, bconst, b_is_array, st))) return rc;
        if ((rc = enqueue_ratio(Pb, 3, st))) return rc;
    }
    return SGP_OK;
}

// One RL round (Eq.1/13/21): q_j = A_j f and J0(f(k)) with the stopping rules, then the multiplicative update.
template <typename T>
int PlanImpl<T>::enqueue_rl_round(const DevOpts &o, const Trace &tr, const double *bconst, int b_is_array, cudaStream_t st)
{
    int rc;
    RowParams<T> Pb = row_params();
    Pb.o = o; Pb.tr = tr; Pb.check_status = 1; Pb.b_is_array = b_is_array;
    for (int j = 0; j < p; ++j) Pb.bconst[j] = bconst[j];
    cur_slot = SGP_PROF_R1;
    { RowParams<T> P = Pb; P.in0 = f; P.maskmode = MM_NONE; if ((rc = launch_row(k_rowf[RF_PLAIN], P, 1, st))) return rc; }
    cur_slot = SGP_PROF_R2;
    { ColParams<T> Q = col_params(); Q.check_status = 1; if ((rc = launch_col(k_mult_run, Q, st))) return rc; }
    cur_slot = SGP_PROF_R3;
    { RowParams<T> P = Pb; P.submode = QJ_RL; P.in0 = Gp; P.in2 = Bp; P.out0 = q; P.part = part_J; if ((rc = launch_row(k_rowi[RI_QJ], P, p, st))) return rc; }
    cur_slot = SGP_PROF_R4;
    { RowParams<T> P = Pb; P.in0 = Gp; P.in1 = q; P.in2 = Bp; if ((rc = launch_row(k_rowf[RF_RATIO], P, p, st))) return rc; }
    cur_slot = SGP_PROF_R5;
    { ColParams<T> Q = col_params(); Q.check_status = 1; if ((rc = launch_col(k_conj_run, Q, st))) return rc; }
    cur_slot = SGP_PROF_R6;
    { RowParams<T> P = Pb; P.in0 = f; P.out0 = f; if ((rc = launch_row(k_rowi[RI_RLUPDATE], P, 1, st))) return rc; }
    cur_slot = -1;
    return SGP_OK;
}

// One OSEM iteration (Algorithm 2): for j = 1..p, h <- (M_R/alpha_j) o h o A_j^T(g_j / (A_j h + b_j))
// (Eq.15; Eq.22 with boundary-effect correction): the six launches of an RL round restricted to image j -- the
// single-image column kernels with K^_j, scaling 1 instead of 1/p (Geom::p = 1), alpha_j on R in place of alpha.
// 4p two-dimensional FFTs.  h lives in f.
template <typename T>
int PlanImpl<T>::enqueue_osem_cycle(const DevOpts &o, const Trace &tr, const double *bconst, int b_is_array, cudaStream_t st)
{
    int rc;
    RowParams<T> Pb = row_params();
    Pb.o = o; Pb.tr = tr; Pb.check_status = 1; Pb.b_is_array = b_is_array;
    Pb.G.p = 1;
    for (int j = 0; j < p; ++j) {
        const size_t off = (size_t)j * n;
        Pb.bconst[0] = bconst[j];
        Pb.alphaR = G.masked ? alphaJ + off : nullptr;
        ColParams<T> Qb = col_params();
        Qb.check_status = 1; Qb.p = 1; Qb.khat = khat + (size_t)j * nspec; Qb.khatB = khatB + (size_t)j * ny;
        cur_slot = SGP_PROF_R1;
        { RowParams<T> P = Pb; P.in0 = f; P.maskmode = MM_NONE; if ((rc = launch_row(k_rowf[RF_PLAIN], P, 1, st))) return rc; }
        cur_slot = SGP_PROF_R2;
        if ((rc = launch_col(k_mult1, Qb, st))) return rc;
        cur_slot = SGP_PROF_R3;
        { RowParams<T> P = Pb; P.submode = QJ_PLAIN; P.in0 = Gp + off; P.in2 = Bp + off; P.out0 = q + off; P.part = part_J;
          if ((rc = launch_row(k_rowi[RI_QJ], P, 1, st))) return rc; }
        cur_slot = SGP_PROF_R4;
        { RowParams<T> P = Pb; P.in0 = Gp + off; P.in1 = q + off; P.in2 = Bp + off; if ((rc = launch_row(k_rowf[RF_RATIO], P, 1, st))) return rc; }
        cur_slot = SGP_PROF_R5;
        if ((rc = launch_col(k_conj1, Qb, st))) return rc;
        cur_slot = SGP_PROF_R6;
        { RowParams<T> P = Pb; P.in0 = f; P.out0 = f; if ((rc = launch_row(k_rowi[RI_RLUPDATE], P, 1, st))) return rc; }
    }
    cur_slot = -1;
    return SGP_OK;
}

// `count` iterations (SGP), rounds (RL) or cycles (OSEM).  With opt.use_graph the launches of kGraphIters iterations are captured
// once per run into a CUDA graph (on a stream of the plan: the caller's may be the legacy default stream, which
// cannot be captured) and the graph is replayed; everything the kernels branch on lives in the control block, so
// the launch parameters of all iterations are identical.
template <typename T>
int PlanImpl<T>::enqueue_many(int algorithm, int count, const RowParams<T> &Pb, const DevOpts &o, const Trace &tr,
                              const double *bconst, int b_is_array, cudaStream_t st)
{
    int rc;
    auto one = [&](cudaStream_t s) -> int {
        return algorithm == SGP_ALG_SGP ? enqueue_sgp_iteration(Pb, o, tr, bconst, b_is_array, s)
             : algorithm == SGP_ALG_RL  ? enqueue_rl_round(o, tr, bconst, b_is_array, s)
                                        : enqueue_osem_cycle(o, tr, bconst, b_is_array, s);
    };
    constexpr int kGraphIters = 10;
    if ((opt.use_graph & 1) && !profiling && count >= kGraphIters) {
        if (!gexec) {
            if (!cap_stream) SGP_CUDA_TRY(cudaStreamCreateWithFlags(&cap_stream, cudaStreamNonBlocking));
            if (!cap_stream2) SGP_CUDA_TRY(cudaStreamCreateWithFlags(&cap_stream2, cudaStreamNonBlocking));
            if (!ev_fork) SGP_CUDA_TRY(cudaEventCreateWithFlags(&ev_fork, cudaEventDisableTiming));
            if (!ev_join) SGP_CUDA_TRY(cudaEventCreateWithFlags(&ev_join, cudaEventDisableTiming));
            cudaGraph_t g = nullptr;
            const long l0 = launches;
            SGP_CUDA_TRY(cudaStreamBeginCapture(cap_stream, cudaStreamCaptureModeThreadLocal));
            rc = SGP_OK;
            for (int i = 0; i < kGraphIters && !rc; ++i) rc = one(cap_stream);
            cudaError_t e = cudaStreamEndCapture(cap_stream, &g);
            graph_launches = launches - l0; launches = l0;
            if (rc) { if (g) cudaGraphDestroy(g); return rc; }
            SGP_CUDA_TRY(e);
            e = cudaGraphInstantiate(&gexec, g, 0);
            cudaGraphDestroy(g);
            SGP_CUDA_TRY(e);
        }
        while (count >= kGraphIters) { SGP_CUDA_TRY(cudaGraphLaunch(gexec, st)); count -= kGraphIters; launches += graph_launches; }
    }
    for (int i = 0; i < count; ++i) if ((rc = one(st))) return rc;
    return SGP_OK;
}

template <typename T>
int PlanImpl<T>::run(int algorithm, const void *const *g, const void *const *b_arr, const double *b_const,
                     const void *f0, void *f_out, const sgp_options *ropt, sgp_result *res, cudaStream_t st)
{
    if (!psf_set || !g || !f_out || !res) return SGP_ERR_ARG;
    if (!b_arr && !b_const) return SGP_ERR_ARG;
    if (algorithm != SGP_ALG_SGP && algorithm != SGP_ALG_RL && algorithm != SGP_ALG_OSEM) return SGP_ERR_ARG;
    sgp_options ro = ropt ? *ropt : opt;
    int rc = validate_options(&ro);
    if (rc) return rc;
    if (ro.refresh_every != 0) return SGP_ERR_UNSUPPORTED;
    if (algorithm == SGP_ALG_OSEM && ro.stop_rule != SGP_STOP_MAXIT) return SGP_ERR_UNSUPPORTED;   // include/sgp.h: osem_*
    if (ro.init == SGP_INIT_USER && !f0) return SGP_ERR_ARG;
    for (int j = 0; j < p; ++j) if (!g[j]) return SGP_ERR_ARG;
    int b_is_array = 0;
    double bconst[kMaxP] = {0};
    for (int j = 0; j < p; ++j) {
        const bool arr = b_arr && b_arr[j];
        if (j == 0) b_is_array = arr ? 1 : 0;
        else if ((arr ? 1 : 0) != b_is_array) return SGP_ERR_ARG;     // all arrays or all constants
        if (!arr) { if (!b_const) return SGP_ERR_ARG; bconst[j] = b_const[j]; }
    }
    const long launches0 = launches;
    if (profiling) prof_reset();
    // Column product kernels of this run.  The two-CTAs-per-SM form (col2_kernel) is 25-30 % faster where the tiles
    // make several waves (4096^2: 82 -> 58 us per pass); at 2048^2 its single wave (all CTAs load, transform and store
    // in phase) loses to the one-CTA form with the TMA-staged transfer function (SGP: 31 vs 23 us; RL: 24 vs 21 us).
    {
        const bool use2 = col2 && ntiles > 2 * nsm;
        k_conj_run = use2 ? k_conj2 : k_conj;
        k_mult_run = use2 ? k_mult2 : k_mult;
    }

    DevOpts o;
    memset(&o, 0, sizeof(o));
    o.beta = ro.beta; o.theta = ro.theta; o.alpha0 = ro.alpha0; o.alpha_min = ro.alpha_min; o.alpha_max = ro.alpha_max;
    o.tol = ro.tol; o.disc_threshold = ro.disc_threshold; o.m_alpha = ro.m_alpha; o.alt_start = ro.alt_start;
    o.armijo_memory = ro.armijo_memory; o.max_iter = ro.max_iter; o.stop_rule = ro.stop_rule;
    o.max_backtracks = ro.max_backtracks; o.adaptive_L = ro.adaptive_L; o.p = p;
    o.nS_total = (double)p * (double)G.sy * (double)G.sx;
    o.rl_relax = algorithm == SGP_ALG_RL ? ro.rl_relax : 1.0;      // Eq.3 is a variant of RL (Eq.1/13/21) only
    o.rl_linear = algorithm == SGP_ALG_RL ? ro.rl_linear : 1.0;    // and so is Eq.4

    Trace tr;
    if ((rc = ensure_trace(ro.max_iter, res, &tr, st))) return rc;

    // ---- start-point phase (a0''): clean inputs, f(0), q_j = A_j f(0), J0(f(0)), adaptive bounds
    SGP_CUDA_TRY(cudaEventRecord(ev0, st));
    Ctrl h;
    memset(&h, 0, sizeof(h));
    h.alpha_prev = ro.alpha0; h.tau = ro.tau1; h.L1 = ro.L1; h.L2 = ro.L2; h.lambda = 1.0;
    h.qsel = 0; h.need_k1 = 1; h.accepted = 1;
    SGP_CUDA_TRY(cudaMemcpyAsync(ct, &h, sizeof(Ctrl), cudaMemcpyHostToDevice, st));
    SGP_CUDA_TRY(cudaMemsetAsync(q + n * (size_t)p, 0, sizeof(T) * n * (size_t)p, st));     // second q buffer: zero outside S
    const int eg = ew_grid(n) > 1024 ? 1024 : ew_grid(n);
    for (int j = 0; j < p; ++j) {
        embed_inputs_kernel<T><<<eg, 256, 0, st>>>((const T *)g[j], b_is_array ? (const T *)b_arr[j] : nullptr, Gp + (size_t)j * n,
                                                   b_is_array ? Bp + (size_t)j * n : nullptr, G, bconst[j], ro.strict, ct,
                                                   part_misc + (size_t)j * 1024);
        launches++;
        if (eg < 1024) SGP_CUDA_TRY(cudaMemsetAsync(part_misc + (size_t)j * 1024 + eg, 0, sizeof(double) * (1024 - eg), st));
    }
    const_start_kernel<T><<<1, 32, 0, st>>>(part_misc, 1024 * p, o.nS_total, ct);
    launches++;
    start_point_kernel<T><<<ew_grid(n), 256, 0, st>>>(f, (const T *)f0, Gp, alphaR, G, ro.init, ct);
    launches++;
    SGP_CUDA_TRY(cudaGetLastError());

    RowParams<T> Pb = row_params();
    Pb.o = o; Pb.tr = tr; Pb.check_status = 1; Pb.b_is_array = b_is_array;
    for (int j = 0; j < p; ++j) Pb.bconst[j] = bconst[j];

    if (algorithm == SGP_ALG_SGP) {
        { RowParams<T> P = Pb; P.in0 = f; if ((rc = launch_row(k_rowf[RF_PLAIN], P, 1, st))) return rc; }
        { ColParams<T> Q = col_params(); Q.check_status = 1; if ((rc = launch_col(k_mult_run, Q, st))) return rc; }
        { RowParams<T> P = Pb; P.submode = QJ_INIT; P.in0 = Gp; P.in2 = Bp; P.out0 = q; P.part = part_J;
          if ((rc = launch_row(k_rowi[RI_QJ], P, p, st))) return rc; }
        if (ro.adaptive_L) {     // bounds from one RL step
            { RowParams<T> P = Pb; P.in0 = Gp; P.in1 = q; P.in2 = Bp; if ((rc = launch_row(k_rowf[RF_RATIO], P, p, st))) return rc; }
            { ColParams<T> Q = col_params(); Q.check_status = 1; if ((rc = launch_col(k_conj_run, Q, st))) return rc; }
            { RowParams<T> P = Pb; P.submode = RIP_RLMINMAX; P.in0 = f; P.part = part_J; if ((rc = launch_row(k_rowi[RI_PLAIN], P, 1, st))) return rc; }
        }
    }
    SGP_CUDA_TRY(cudaEventRecord(ev1, st));
    SGP_CUDA_TRY(cudaMemcpyAsync(&h, ct, sizeof(Ctrl), cudaMemcpyDeviceToHost, st));
    SGP_CUDA_TRY(cudaStreamSynchronize(st));
    int status = h.status;
    if (h.flag_data & 1) status = SGP_ERR_DATA;
    else if (h.flag_data & 2) status = SGP_ERR_DATA;
    else if (h.flag_data & 4) status = SGP_ERR_DATA;

    // ---- iteration loop
    long fft2 = 0;
    if (status == 0) {
        int chunk = ro.check_every > 0 ? ro.check_every : (ro.stop_rule == SGP_STOP_MAXIT ? 200 : 20);
        if (algorithm == SGP_ALG_SGP) {
            if (ro.max_iter == 0) status = SGP_REASON_MAXIT;
            else if ((rc = enqueue_ratio(Pb, 3, st))) return rc;        // K1 of iteration 0; every iteration enqueues the next one's
            int done = 0;
            while (status == 0) {
                int todo = ro.max_iter - done; if (todo > chunk) todo = chunk;
                if (todo < 1) { status = SGP_REASON_MAXIT; break; }
                if ((rc = enqueue_many(algorithm, todo, Pb, o, tr, bconst, b_is_array, st))) return rc;
                SGP_CUDA_TRY(cudaMemcpyAsync(&h, ct, sizeof(Ctrl), cudaMemcpyDeviceToHost, st));
                SGP_CUDA_TRY(cudaStreamSynchronize(st));
                status = h.status; done = h.k;
                if (status == 0 && done >= ro.max_iter) status = SGP_REASON_MAXIT;   // not reachable: the device sets it
            }
            fft2 = (long)h.k * (2 * p + 2);
        } else if (algorithm == SGP_ALG_OSEM) {
            // max_iter cycles, then J0 (Eq.12) at the final iterate: q_j = A_j f for all j, as in the start-point phase
            int done = 0;
            while (status == 0 && done < ro.max_iter) {
                int todo = ro.max_iter - done; if (todo > chunk) todo = chunk;
                if ((rc = enqueue_many(algorithm, todo, Pb, o, tr, bconst, b_is_array, st))) return rc;
                done += todo;
                SGP_CUDA_TRY(cudaMemcpyAsync(&h, ct, sizeof(Ctrl), cudaMemcpyDeviceToHost, st));
                SGP_CUDA_TRY(cudaStreamSynchronize(st));
                status = h.status;
            }
            fft2 = (long)done * 4 * p;
            if (status == 0) {
                Trace t0 = tr; t0.J = nullptr;
                RowParams<T> Pj = Pb; Pj.tr = t0;
                { RowParams<T> P = Pj; P.in0 = f; if ((rc = launch_row(k_rowf[RF_PLAIN], P, 1, st))) return rc; }
                { ColParams<T> Q = col_params(); Q.check_status = 1; if ((rc = launch_col(k_mult_run, Q, st))) return rc; }
                { RowParams<T> P = Pj; P.submode = QJ_INIT; P.in0 = Gp; P.in2 = Bp; P.out0 = q; P.part = part_J;
                  if ((rc = launch_row(k_rowi[RI_QJ], P, p, st))) return rc; }
                SGP_CUDA_TRY(cudaMemcpyAsync(&h, ct, sizeof(Ctrl), cudaMemcpyDeviceToHost, st));
                SGP_CUDA_TRY(cudaStreamSynchronize(st));
                status = h.status;
                h.k = done;
                if (status == 0) status = SGP_REASON_MAXIT;
            }
        } else {
            int rounds = 0;     // round k evaluates J0(f(k)) and, unless a rule fires, makes update k+1
            while (status == 0) {
                int todo = ro.max_iter + 1 - rounds; if (todo > chunk) todo = chunk; if (todo < 1) todo = 1;
                if ((rc = enqueue_many(algorithm, todo, Pb, o, tr, bconst, b_is_array, st))) return rc;
                rounds += todo;
                SGP_CUDA_TRY(cudaMemcpyAsync(&h, ct, sizeof(Ctrl), cudaMemcpyDeviceToHost, st));
                SGP_CUDA_TRY(cudaStreamSynchronize(st));
                status = h.status;
            }
            fft2 = (long)h.k * (2 * p + 2) + (p + 1);
        }
    }
    SGP_CUDA_TRY(cudaEventRecord(ev2, st));
    if (gexec) { cudaGraphExecDestroy(gexec); gexec = nullptr; }      // the kernels it holds are already enqueued
    final_update_kernel<T><<<ew_grid(n), 256, 0, st>>>(f, d, (T *)f_out, n, ct);     // a10: the last accepted step, if still pending
    launches++;
    SGP_CUDA_TRY(cudaGetLastError());
    const int kdone = h.k;
    if (res->trace_J) SGP_CUDA_TRY(cudaMemcpyAsync(res->trace_J, trJ, sizeof(double) * (kdone + 1), cudaMemcpyDeviceToHost, st));
    if (kdone > 0) {
        if (res->trace_alpha) SGP_CUDA_TRY(cudaMemcpyAsync(res->trace_alpha, trA, sizeof(double) * kdone, cudaMemcpyDeviceToHost, st));
        if (res->trace_lambda) SGP_CUDA_TRY(cudaMemcpyAsync(res->trace_lambda, trL, sizeof(double) * kdone, cudaMemcpyDeviceToHost, st));
        if (res->trace_rule) SGP_CUDA_TRY(cudaMemcpyAsync(res->trace_rule, trR, sizeof(int) * kdone, cudaMemcpyDeviceToHost, st));
        if (res->trace_backtracks) SGP_CUDA_TRY(cudaMemcpyAsync(res->trace_backtracks, trB, sizeof(int) * kdone, cudaMemcpyDeviceToHost, st));
    }
    SGP_CUDA_TRY(cudaStreamSynchronize(st));
    if (profiling) prof_collect();
    float ms01 = 0.f, ms12 = 0.f;
    cudaEventElapsedTime(&ms01, ev0, ev1);
    cudaEventElapsedTime(&ms12, ev1, ev2);
    res->iterations = kdone;
    res->stop_reason = status > 0 ? status : 0;
    res->J0_final = h.J;
    res->discrepancy_final = 2.0 * h.J / o.nS_total;
    res->total_backtracks = h.total_backtracks;
    res->L1_used = algorithm == SGP_ALG_SGP ? h.L1 : 0.0;
    res->L2_used = algorithm == SGP_ALG_SGP ? h.L2 : 0.0;
    res->n_fft2 = fft2;
    res->setup_ms = ms01; res->loop_ms = ms12;
    res->kernel_launches = launches - launches0;
    res->fused_linesearch = (algorithm == SGP_ALG_SGP && fuse_ls) ? 1 : 0;
    return status < 0 ? status : SGP_OK;
}

PlanBase *SGP_MAKE() { return new PlanImpl<SGP_T>(); }

}  // namespace sgpk
