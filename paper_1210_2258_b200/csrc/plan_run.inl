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
    const int need = max_iter + 2;
    const size_t per = 6 * sizeof(double) + 2 * sizeof(int);
    if (need > trace_cap) {
        free_trace();
        const size_t cap = ((size_t)need + 1) & ~(size_t)1;     // even: the int arrays stay 8-byte aligned
        SGP_CUDA_TRY(cudaMalloc((void **)&trJ, per * cap * (size_t)nb));      // one block per problem, one allocation
        trA = trJ + cap; trL = trA + cap; fA = trL + cap; fL = fA + cap; trE = fL + cap;
        trR = reinterpret_cast<int *>(trE + cap); trB = trR + cap;
        trace_cap = (int)cap;
    }
    tr_slab = nb > 1 ? per * (size_t)trace_cap : 0;
    SGP_CUDA_TRY(cudaMemsetAsync(trJ, 0, per * (size_t)trace_cap * (size_t)nb, st));
    tr->J = trJ; tr->alpha = trA; tr->lambda = trL; tr->rule = trR; tr->backtracks = trB;
    tr->force_alpha = nullptr; tr->force_lambda = nullptr;
    tr->err = res->truth ? trE : nullptr;
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
// u_j + J(lambda = 1) + Armijo test + book-keeping (fused form: also q(k+1), the ratio and its row FFT), then
// K1 = [Armijo backtracking, only after a rejected lambda = 1] + ratio + row FFT of iteration k + 1 (returns at once when
// the fused K6 has already done its work).  Six launches; the ratio kernel of the FIRST iteration is enqueued by run().
template <typename T>
int PlanImpl<T>::enqueue_ratio(const RowParams<T> &Pb, int lazy, cudaStream_t st)
{
    cur_slot = SGP_PROF_K1;
    RowParams<T> P = Pb; P.lazy = lazy; P.in0 = Gp; P.in1 = q; P.in2 = Bp; P.in3 = u; P.out0 = q;
    P.btinfo = btinfo;
    int rc = launch_row(k_rowf[RF_RATIO], P, p, st);
    cur_slot = -1;
    return rc;
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
        P.count_fft = p + 1; if ((rc = launch_row(k_rowi[RI_GRAD], P, 1, st))) return rc;
    }
    if (o.flux_constraint) {   // the multiplier mu of the flux-constrained projection (extra.cuh): Newton steps, no FFT
        flux_arm_kernel<0><<<1, 32, 0, st>>>(fxsync, ct);
        FluxParams<T> F;
        memset(&F, 0, sizeof(F));
        F.G = G; F.ct = ct; F.f = f; F.grad = grad; F.alphaR = alphaR; F.part = part_fx; F.sync = fxsync;
        F.nchunks = (unsigned int)fx_chunks; F.chunk_batches = (unsigned int)fx_batches; F.max_rounds = 100;
        const int fg = (int)(fx_chunks < (size_t)(2 * nsm) ? fx_chunks : (size_t)(2 * nsm));
        flux_mu_kernel<T><<<fg, 256, 0, st>>>(F);
        launches += 2;
        SGP_CUDA_TRY(cudaGetLastError());
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
        RowParams<T> P = Pb; P.in0 = Gp; P.in1 = q; P.in2 = Bp; P.out0 = u; P.part = part_J; P.part2 = part_gd; P.btsync = btsync;
        P.count_fft = p + 1; if ((rc = launch_row(k_rowi[fuse_ls ? RI_LSF : RI_LS], P, p, st))) return rc;
    }
    cur_slot = -1;
    // ---- tail: K1 of the next iteration (a9 for lambda < 1 as its prologue, a11, a10 for q, a1)
    if ((rc = enqueue_ratio(Pb, 1, st))) return rc;
    if (tr.err) {      // Eq.25: error of the step just accepted; with SGP_STOP_MINERR an increase discards it (extra.cuh)
        err_kernel<T><<<ew_grid(n), 256, 0, st>>>(f, d, nullptr, (const T *)run_truth, n, ct, o, tr, part_err, 1);
        launches++;
        SGP_CUDA_TRY(cudaGetLastError());
    }
    if (o.refresh_every > 0) {
        // reading A21: after every refresh_every-th iteration q_j = A_j f(k+1) and J0 are recomputed from f (the kernels of
        // this round return at once otherwise): apply the pending step to f, row FFT of f, column pass x K^_j, inverse rows
        // -> q_j, J0, stopping rules; then the ratio of the next iteration once more, from the recomputed q
        apply_pending_kernel<T><<<ew_grid(n), 256, 0, st>>>(f, d, n, ct);
        refresh_flags_kernel<0><<<1, 32, 0, st>>>(ct, ct_shadow);
        launches += 2;
        SGP_CUDA_TRY(cudaGetLastError());
        { RowParams<T> P = Pb; P.in0 = f; P.lazy = 4; if ((rc = launch_row(k_rowf[RF_PLAIN], P, 1, st))) return rc; }
        { ColParams<T> Q = col_params(); Q.check_status = 1; Q.ct = ct_shadow; if ((rc = launch_col(k_mult_run, Q, st))) return rc; }     // counted by the QJ_REFRESH kernel
        { RowParams<T> P = Pb; P.submode = QJ_REFRESH; P.in0 = Gp; P.in2 = Bp; P.out0 = q; P.part = part_J;
          P.count_fft = p + 1; if ((rc = launch_row(k_rowi[RI_QJ], P, p, st))) return rc; }
        if ((rc = enqueue_ratio(Pb, 2, st))) return rc;
    }
    return SGP_OK;
}

// One RL round (Eq.1/13/21) on the schedule of SURVEY.md 8(d) ("RL schedule", 7p + 6 planes), four launches:
//   R2 column pass x K^_j                       (spectrum of f -> p spectra of A_j f)
//   R3 row C2R -> J0(f(k)), stopping rules -> ratio g_j/(A_j f + b_j) -> row R2C        (RI_QJF; A_j f is never stored)
//   R5 column pass sum_j conj(K^_j)
//   R6 row C2R -> multiplicative update (Eq.1/13/21, Eq.3, Eq.4) -> row R2C of f(k+1)   (RI_RLUPF)
// The row transform of f(0) (R1) is enqueued once by run().  `fused = false` (opt.use_graph bit 6, and the Eq.25 rule,
// which must see f(k+1) before it replaces f(k)) keeps the six separate launches of round 1.
template <typename T>
int PlanImpl<T>::enqueue_rl_round(const DevOpts &o, const Trace &tr, const double *bconst, int b_is_array, cudaStream_t st)
{
    int rc;
    RowParams<T> Pb = row_params();
    Pb.o = o; Pb.tr = tr; Pb.check_status = 1; Pb.b_is_array = b_is_array;
    for (int j = 0; j < p; ++j) Pb.bconst[j] = bconst[j];
    if (!rl_fused) {
        cur_slot = SGP_PROF_R1;
        { RowParams<T> P = Pb; P.in0 = f; P.maskmode = MM_NONE; if ((rc = launch_row(k_rowf[RF_PLAIN], P, 1, st))) return rc; }
    }
    cur_slot = SGP_PROF_R2;
    { ColParams<T> Q = col_params(); Q.check_status = 1; if ((rc = launch_col(k_mult_run, Q, st))) return rc; }
    cur_slot = SGP_PROF_R3;
    if (rl_fused) {
        RowParams<T> P = Pb; P.submode = QJ_RL; P.in0 = Gp; P.in2 = Bp; P.part = part_J;
        P.count_fft = p + 1; if ((rc = launch_row(k_rowi[RI_QJF], P, p, st))) return rc;
    } else {
        { RowParams<T> P = Pb; P.submode = QJ_RL; P.in0 = Gp; P.in2 = Bp; P.out0 = q; P.part = part_J; P.count_fft = p + 1; if ((rc = launch_row(k_rowi[RI_QJ], P, p, st))) return rc; }
        cur_slot = SGP_PROF_R4;
        { RowParams<T> P = Pb; P.in0 = Gp; P.in1 = q; P.in2 = Bp; if ((rc = launch_row(k_rowf[RF_RATIO], P, p, st))) return rc; }
    }
    cur_slot = SGP_PROF_R5;
    { ColParams<T> Q = col_params(); Q.check_status = 1; if ((rc = launch_col(k_conj_run, Q, st))) return rc; }
    cur_slot = SGP_PROF_R6;
    if (tr.err) {
        // Eq.25: the update goes to the plane `d` (unused by RL), its error is evaluated, and it replaces f only if the
        // rule lets it (extra.cuh); needs the separate kernels (rl_fused is off)
        { RowParams<T> P = Pb; P.in0 = f; P.out0 = d; P.count_fft = p + 1; if ((rc = launch_row(k_rowi[RI_RLUPDATE], P, 1, st))) return rc; }
        err_kernel<T><<<ew_grid(n), 256, 0, st>>>(f, nullptr, d, (const T *)run_truth, n, ct, o, tr, part_err, 2);
        rl_commit_kernel<T><<<ew_grid(n), 256, 0, st>>>(f, d, n, ct);
        launches += 2;
        SGP_CUDA_TRY(cudaGetLastError());
    } else {
        RowParams<T> P = Pb; P.in0 = f; P.out0 = f;
        P.count_fft = p + 1; if ((rc = launch_row(k_rowi[rl_fused ? RI_RLUPF : RI_RLUPDATE], P, 1, st))) return rc;
    }
    cur_slot = -1;
    return SGP_OK;
}

// One OSEM iteration (Algorithm 2): for j = 1..p, h <- (M_R/alpha_j) o h o A_j^T(g_j / (A_j h + b_j))
// (Eq.15; Eq.22 with boundary-effect correction): the launches of an RL round restricted to image j -- the
// single-image column kernels with K^_j, scaling 1 instead of 1/p (Geom::p = 1), alpha_j on R in place of alpha.
// 4p two-dimensional FFTs.  h lives in f.
template <typename T>
int PlanImpl<T>::enqueue_osem_cycle(const DevOpts &o, const Trace &tr, const double *bconst, int b_is_array, cudaStream_t st)
{
    int rc;
    RowParams<T> Pb = row_params();
    Pb.o = o; Pb.tr = tr; Pb.check_status = 1; Pb.b_is_array = b_is_array;
    Pb.G.p = 1;
    if (tr.err) {      // Eq.25 per cycle (reading A27): h(k) is kept in `d` until the error of h(k+1) is known (extra.cuh)
        osem_backup_kernel<T><<<ew_grid(n), 256, 0, st>>>(f, d, n, ct);
        launches++;
        SGP_CUDA_TRY(cudaGetLastError());
    }
    for (int j = 0; j < p; ++j) {
        const size_t off = (size_t)j * n;
        Pb.bconst[0] = bconst[j];
        Pb.alphaR = G.masked ? alphaJ + off : nullptr;
        ColParams<T> Qb = col_params();
        Qb.check_status = 1; Qb.p = 1; Qb.khat = khat + (size_t)j * nspec; Qb.khatB = khatB + (size_t)j * ny;
        if (!rl_fused) {
            cur_slot = SGP_PROF_R1;
            { RowParams<T> P = Pb; P.in0 = f; P.maskmode = MM_NONE; if ((rc = launch_row(k_rowf[RF_PLAIN], P, 1, st))) return rc; }
        }
        cur_slot = SGP_PROF_R2;
        if ((rc = launch_col(k_mult1, Qb, st))) return rc;
        cur_slot = SGP_PROF_R3;
        if (rl_fused) {
            RowParams<T> P = Pb; P.submode = QJ_PLAIN; P.in0 = Gp + off; P.in2 = Bp + off; P.part = part_J;
            P.count_fft = 2; if ((rc = launch_row(k_rowi[RI_QJF], P, 1, st))) return rc;
        } else {
            { RowParams<T> P = Pb; P.submode = QJ_PLAIN; P.in0 = Gp + off; P.in2 = Bp + off; P.out0 = q + off; P.part = part_J;
              P.count_fft = 2; if ((rc = launch_row(k_rowi[RI_QJ], P, 1, st))) return rc; }
            cur_slot = SGP_PROF_R4;
            { RowParams<T> P = Pb; P.in0 = Gp + off; P.in1 = q + off; P.in2 = Bp + off; if ((rc = launch_row(k_rowf[RF_RATIO], P, 1, st))) return rc; }
        }
        cur_slot = SGP_PROF_R5;
        if ((rc = launch_col(k_conj1, Qb, st))) return rc;
        cur_slot = SGP_PROF_R6;
        { RowParams<T> P = Pb; P.in0 = f; P.out0 = f; P.count_fft = 2; if ((rc = launch_row(k_rowi[rl_fused ? RI_RLUPF : RI_RLUPDATE], P, 1, st))) return rc; }
    }
    cur_slot = -1;
    if (tr.err) {
        err_kernel<T><<<ew_grid(n), 256, 0, st>>>(f, nullptr, nullptr, (const T *)run_truth, n, ct, o, tr, part_err, 3);
        osem_restore_kernel<T><<<ew_grid(n), 256, 0, st>>>(f, d, n, ct);
        launches += 2;
        SGP_CUDA_TRY(cudaGetLastError());
    }
    return SGP_OK;
}

// `count` iterations (SGP), rounds (RL) or cycles (OSEM).  With opt.use_graph the launches of kGraphIters iterations are captured
// into a CUDA graph (on a stream of the plan: the caller's may be the legacy default stream, which cannot be captured)
// and the graph is replayed; everything the kernels branch on lives in the control block, so the launch parameters of
// all iterations are identical.  The instantiated graph is KEPT across run() calls and re-used as long as the launch
// parameters are the same (`sig`: algorithm, device options, trace pointers, backgrounds, schedule switches).
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
    if (run_graph && !profiling && count >= kGraphIters) {
        GraphSig sig;
        memset(&sig, 0, sizeof(sig));
        sig.algorithm = algorithm; sig.b_is_array = b_is_array;
        memcpy(&sig.o, &o, sizeof(o)); memcpy(&sig.tr, &tr, sizeof(tr));
        for (int j = 0; j < p; ++j) sig.bconst[j] = bconst[j];
        sig.truth = run_truth; sig.fuse_ls = fuse_ls; sig.rl_fused = rl_fused; sig.k_conj = (const void *)k_conj_run; sig.k_mult = (const void *)k_mult_run;
        if (gexec && memcmp(&sig, &gsig, sizeof(sig)) != 0) { cudaGraphExecDestroy(gexec); gexec = nullptr; }
        if (!gexec) {
            if (!cap_stream) SGP_CUDA_TRY(cudaStreamCreateWithFlags(&cap_stream, cudaStreamNonBlocking));
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
            if (e != cudaSuccess) gexec = nullptr;
            SGP_CUDA_TRY(e);
            memcpy(&gsig, &sig, sizeof(sig));
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
    if (nb != 1) return SGP_ERR_ARG;             // a batched plan runs through sgp_plan_run_batched
    const void *f0s[1] = {f0};
    void *fouts[1] = {f_out};
    return run_batched(algorithm, g, b_arr, b_const, f0 ? f0s : nullptr, f_out ? fouts : nullptr, ropt, res, st);
}

// nb problems of the plan's geometry at once (nb = 1: an ordinary run).  g, b_arr, b_const: nb * p entries, problem-major
// (problem b, image j at b * p + j); f0, f_out, res: nb entries.  Every kernel of the iteration is launched once for all
// problems (blockIdx.z = problem); each problem has its own control block, so step lengths, backtracking and stopping
// are per problem, and a problem that has stopped costs nothing more than the early return of its CTAs.
template <typename T>
int PlanImpl<T>::run_batched(int algorithm, const void *const *g, const void *const *b_arr, const double *b_const,
                             const void *const *f0, void *const *f_out, const sgp_options *ropt, sgp_result *res, cudaStream_t st)
{
    if (!psf_set || !g || !f_out || !res) return SGP_ERR_ARG;
    if (!b_arr && !b_const) return SGP_ERR_ARG;
    if (algorithm != SGP_ALG_SGP && algorithm != SGP_ALG_RL && algorithm != SGP_ALG_OSEM) return SGP_ERR_ARG;
    sgp_options ro = ropt ? *ropt : opt;
    int rc = validate_options(&ro);
    if (rc) return rc;
    if (algorithm == SGP_ALG_OSEM && ro.stop_rule != SGP_STOP_MAXIT && ro.stop_rule != SGP_STOP_MINERR) return SGP_ERR_UNSUPPORTED;   // include/sgp.h: osem_*
    if (ro.stop_rule == SGP_STOP_MINERR && !res[0].truth) return SGP_ERR_ARG;                       // Eq.25 needs the true object
    // plan-level fields cannot change per run (include/sgp.h: sgp_plan_run)
    if (ro.tile_cols != opt.tile_cols || ro.rows_per_block != opt.rows_per_block || ro.sigma_R != opt.sigma_R ||
        ro.psf_origin != opt.psf_origin || ((ro.use_graph ^ opt.use_graph) & ~1)) return SGP_ERR_ARG;
    if (nb > 1) {     // not available for batched plans (include/sgp.h: sgp_plan_create_batched)
        if (ro.flux_constraint || ro.refresh_every || ro.stop_rule == SGP_STOP_MINERR || (ro.init == SGP_INIT_CONST_SMOOTH && G.masked))
            return SGP_ERR_UNSUPPORTED;
        for (int b = 0; b < nb; ++b) if (res[b].truth || res[b].force_alpha || res[b].force_lambda) return SGP_ERR_UNSUPPORTED;
    }
    struct LaunchWidth { int &v; int old; LaunchWidth(int &v_, int n) : v(v_), old(v_) { v = n; } ~LaunchWidth() { v = old; } } lw(lnb, nb);
    run_graph = (ro.use_graph & 1) != 0;
    run_truth = res[0].truth;
    rl_fused = !(opt.use_graph & 64) && !(algorithm == SGP_ALG_RL && run_truth);
    if (ro.init == SGP_INIT_USER && !f0) return SGP_ERR_ARG;
    for (int b = 0; b < nb; ++b) {
        if (!f_out[b] || (ro.init == SGP_INIT_USER && !f0[b])) return SGP_ERR_ARG;
        for (int j = 0; j < p; ++j) if (!g[b * p + j]) return SGP_ERR_ARG;
    }
    int b_is_array = 0;
    std::vector<double> bconst_all((size_t)nb * kMaxP, 0.0);
    for (int b = 0; b < nb; ++b)
        for (int j = 0; j < p; ++j) {
            const bool arr = b_arr && b_arr[b * p + j];
            if (b == 0 && j == 0) b_is_array = arr ? 1 : 0;
            else if ((arr ? 1 : 0) != b_is_array) return SGP_ERR_ARG;     // all arrays or all constants
            if (!arr) { if (!b_const) return SGP_ERR_ARG; bconst_all[(size_t)b * kMaxP + j] = b_const[b * p + j]; }
        }
    const double *bconst = bconst_all.data();        // problem 0 (what an ordinary plan's kernels read from their parameters)
    const long launches0 = launches;
    if (profiling) prof_reset();
    // Column product kernels of this run.  The two-CTAs-per-SM form (col2_kernel) is 25-30 % faster where the tiles
    // make several waves (4096^2: 82 -> 58 us per pass); at 2048^2 its single wave (all CTAs load, transform and store
    // in phase) loses to the one-CTA form with the TMA-staged transfer function (SGP: 31 vs 23 us; RL: 24 vs 21 us).
    {
        const bool use2 = col2 && ((size_t)ntiles * nb > 2 * (size_t)nsm || getenv("SGP_FORCE_COL2") != nullptr);
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
    o.flux_constraint = algorithm == SGP_ALG_SGP ? ro.flux_constraint : 0;
    o.refresh_every = algorithm == SGP_ALG_SGP ? ro.refresh_every : 0;

    Trace tr;
    if ((rc = ensure_trace(ro.max_iter, res, &tr, st))) return rc;
    auto pp = [&](auto *ptr, int b) { return bshift_host(ptr, (size_t)b * slab); };      // problem b's copy of a per-problem array

    // ---- start-point phase (a0''): clean inputs, f(0), q_j = A_j f(0), J0(f(0)), adaptive bounds
    SGP_CUDA_TRY(cudaEventRecord(ev0, st));
    std::vector<Ctrl> hs((size_t)nb);
    const int eg = ew_grid(n) > 1024 ? 1024 : ew_grid(n);
    for (int b = 0; b < nb; ++b) {
        Ctrl &h = hs[b];
        memset(&h, 0, sizeof(h));
        h.alpha_prev = ro.alpha0; h.tau = ro.tau1; h.L1 = ro.L1; h.L2 = ro.L2; h.lambda = 1.0;
        h.qsel = 0; h.need_k1 = 1; h.accepted = 1;
        for (int j = 0; j < p; ++j) h.bconst[j] = bconst_all[(size_t)b * kMaxP + j];
    }
    BatchTab tab;
    memset(&tab, 0, sizeof(tab));
    if (nb > 1) {
        // Batched plans: one copy, one memset and one launch per set-up step for ALL problems (blockIdx.z = problem), not one per
        // problem -- with 64 problems of 256^2 the per-problem form spent 5.3 ms in ~600 small copies and launches, as much as
        // 30 of the 100 iterations that followed.  The addresses of the caller's arrays go to the device as one table.
        std::vector<const void *> th((size_t)2 * nb * p + 2 * (size_t)nb, nullptr);
        for (int i = 0; i < nb * p; ++i) { th[i] = g[i]; th[(size_t)nb * p + i] = b_is_array ? b_arr[i] : nullptr; }
        for (int b = 0; b < nb; ++b) { th[(size_t)2 * nb * p + b] = f0 ? f0[b] : nullptr; th[(size_t)2 * nb * p + nb + b] = f_out[b]; }
        SGP_CUDA_TRY(cudaMemcpyAsync(ptrtab, th.data(), th.size() * sizeof(void *), cudaMemcpyHostToDevice, st));
        tab.g = ptrtab; tab.b = ptrtab + (size_t)nb * p; tab.f0 = ptrtab + (size_t)2 * nb * p;
        tab.f_out = (void *const *)(ptrtab + (size_t)2 * nb * p + nb);
        SGP_CUDA_TRY(cudaMemcpy2DAsync(ct, slab, hs.data(), sizeof(Ctrl), sizeof(Ctrl), (size_t)nb, cudaMemcpyHostToDevice, st));
        SGP_CUDA_TRY(cudaMemset2DAsync(q + n * (size_t)p, slab, 0, sizeof(T) * n * (size_t)p, (size_t)nb, st));     // second q buffers: zero outside S
        embed_inputs_batched_kernel<T><<<dim3(eg, p, nb), 256, 0, st>>>(tab, Gp, b_is_array ? Bp : nullptr, G, p, b_is_array, ro.strict, ct, part_misc, slab);
        launches++;
        if (eg < 1024)
            for (int j = 0; j < p; ++j)
                SGP_CUDA_TRY(cudaMemset2DAsync(part_misc + (size_t)j * 1024 + eg, slab, 0, sizeof(double) * (1024 - eg), (size_t)nb, st));
        const_start_batched_kernel<T><<<dim3(1, 1, nb), 32, 0, st>>>(part_misc, 1024 * p, o.nS_total, p, ro.flux_value, ct, slab);
        launches++;
        start_point_batched_kernel<T><<<dim3(ew_grid(n), 1, nb), 256, 0, st>>>(tab, f, Gp, alphaR, G, ro.init == SGP_INIT_CONST_SMOOTH ? SGP_INIT_CONST : ro.init, ct, slab);
        launches++;
    } else {
        const int b = 0;
        SGP_CUDA_TRY(cudaMemcpyAsync(pp(ct, b), &hs[b], sizeof(Ctrl), cudaMemcpyHostToDevice, st));
        SGP_CUDA_TRY(cudaMemsetAsync(pp(q, b) + n * (size_t)p, 0, sizeof(T) * n * (size_t)p, st));     // second q buffer: zero outside S
        for (int j = 0; j < p; ++j) {
            embed_inputs_kernel<T><<<eg, 256, 0, st>>>((const T *)g[b * p + j], b_is_array ? (const T *)b_arr[b * p + j] : nullptr,
                                                       pp(Gp, b) + (size_t)j * n, b_is_array ? pp(Bp, b) + (size_t)j * n : nullptr, G,
                                                       bconst_all[(size_t)b * kMaxP + j], ro.strict, pp(ct, b), pp(part_misc, b) + (size_t)j * 1024);
            launches++;
            if (eg < 1024) SGP_CUDA_TRY(cudaMemsetAsync(pp(part_misc, b) + (size_t)j * 1024 + eg, 0, sizeof(double) * (1024 - eg), st));
        }
        const_start_kernel<T><<<1, 32, 0, st>>>(pp(part_misc, b), 1024 * p, o.nS_total, p, ro.flux_value, pp(ct, b));
        launches++;
        start_point_kernel<T><<<ew_grid(n), 256, 0, st>>>(pp(f, b), f0 ? (const T *)f0[b] : nullptr, pp(Gp, b), alphaR, G,
                                                          ro.init == SGP_INIT_CONST_SMOOTH ? SGP_INIT_CONST : ro.init, pp(ct, b));
        launches++;
    }
    SGP_CUDA_TRY(cudaGetLastError());

    RowParams<T> Pb = row_params();
    Pb.o = o; Pb.tr = tr; Pb.tr_slab = tr_slab; Pb.check_status = 1; Pb.b_is_array = b_is_array;
    for (int j = 0; j < p; ++j) Pb.bconst[j] = bconst[j];

    if (ro.init == SGP_INIT_CONST_SMOOTH && G.masked) {
        // PAPER.md:264, reading A28: f(0) = M_R o max(0, G_sigma * (c M_R)), G_sigma the periodic Gaussian of unit sum.  (Without
        // boundary correction the constant image is its own smoothed version.)  The Gaussian's transfer function goes the
        // way of a PSF (row FFT, column FFT, scaling) into planes that are free during the start-point phase.
        double sy_ = 0.0, sx_ = 0.0;
        for (int y = 0; y < ny; ++y) { const double dy = y <= ny / 2 ? y : y - ny; sy_ += exp(-dy * dy / (2.0 * ro.init_sigma * ro.init_sigma)); }
        for (int x = 0; x < nx; ++x) { const double dx = x <= nx / 2 ? x : x - nx; sx_ += exp(-dx * dx / (2.0 * ro.init_sigma * ro.init_sigma)); }
        gauss_plane_kernel<T><<<ew_grid(n), 256, 0, st>>>(scratch, ny, nx, ro.init_sigma, sy_ * sx_);
        launches++;
        C *khat_tmp = (C *)u;
        { RowParams<T> P = Pb; P.check_status = 0; P.in0 = scratch; P.maskmode = MM_NONE; P.spec = (C *)grad; if ((rc = launch_row(k_rowf[RF_PLAIN], P, 1, st))) return rc; }
        { ColParams<T> Q = col_params(); Q.in = (const C *)grad; Q.out = (C *)grad; if ((rc = launch_col(k_colf, Q, st))) return rc; }
        khat_fixup_kernel<T><<<ew_grid(nspec), 256, 0, st>>>((const C *)grad, khat_tmp, khatB_tmp, ny, nx, G.C);
        launches++;
        SGP_CUDA_TRY(cudaGetLastError());
        { RowParams<T> P = Pb; P.check_status = 0; P.in0 = f; P.maskmode = MM_NONE; if ((rc = launch_row(k_rowf[RF_PLAIN], P, 1, st))) return rc; }
        { ColParams<T> Q = col_params(); Q.khat = khat_tmp; Q.khatB = khatB_tmp; Q.p = 1; if ((rc = launch_col(k_mult1, Q, st))) return rc; }
        { RowParams<T> P = Pb; P.check_status = 0; P.submode = RIP_STORE_POS; P.maskmode = MM_R; P.out0 = f; if ((rc = launch_row(k_rowi[RI_PLAIN], P, 1, st))) return rc; }
    }
    if (o.flux_constraint) {     // reading A26: f(0) rescaled to the flux c
        plane_sum_tmp_kernel<T><<<1, 1024, 0, st>>>(f, n, ct);
        flux_rescale_kernel<T><<<ew_grid(n), 256, 0, st>>>(f, alphaR, n, G, (double)nR, ct);
        launches += 2;
        SGP_CUDA_TRY(cudaGetLastError());
    }
    if (tr.err) {                // Eq.25: rho(0)
        err_kernel<T><<<ew_grid(n), 256, 0, st>>>(f, d, nullptr, (const T *)run_truth, n, ct, o, tr, part_err, 0);
        launches++;
        SGP_CUDA_TRY(cudaGetLastError());
    }

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
    // all control blocks in one strided copy
    auto read_ctrl = [&]() -> int {
        SGP_CUDA_TRY(cudaMemcpy2DAsync(hs.data(), sizeof(Ctrl), ct, slab ? slab : sizeof(Ctrl), sizeof(Ctrl), (size_t)nb, cudaMemcpyDeviceToHost, st));
        SGP_CUDA_TRY(cudaStreamSynchronize(st));
        return SGP_OK;
    };
    if ((rc = read_ctrl())) return rc;
    std::vector<int> status((size_t)nb);
    std::vector<unsigned long long> nfft0((size_t)nb);
    auto any_running = [&]() { for (int b = 0; b < nb; ++b) if (status[b] == 0) return true; return false; };
    for (int b = 0; b < nb; ++b) {
        status[b] = hs[b].status;
        nfft0[b] = hs[b].nfft;                    // transforms of the start-point phase
        if (hs[b].flag_data & 7) status[b] = SGP_ERR_DATA;
    }
    // a problem with bad data must not iterate: its device status is what the kernels test
    for (int b = 0; b < nb; ++b)
        if (status[b] != hs[b].status) SGP_CUDA_TRY(cudaMemcpyAsync(&pp(ct, b)->status, &status[b], sizeof(int), cudaMemcpyHostToDevice, st));

    // small grids: the cluster kernel (small.cuh) for what it covers, the launch-per-pass path for everything else
    const bool small_ok = !b_is_array && ro.stop_rule != SGP_STOP_MINERR && !tr.force_alpha && !tr.force_lambda && !tr.err && !profiling;
    const bool small_run = small_k && small_ok && algorithm == SGP_ALG_SGP && !o.flux_constraint && !o.refresh_every;
    const bool small_rl = small_k_rl && small_ok && algorithm == SGP_ALG_RL;
    if (algorithm == SGP_ALG_SGP && !small_run) {     // arguments of the Armijo backtracking (aux.cuh), read from device memory
        std::vector<BtInfo<T>> bis((size_t)nb);
        for (int b = 0; b < nb; ++b) {
            BtInfo<T> &bi = bis[b];
            memset(&bi, 0, sizeof(bi));
            bi.G = G; bi.o = o; bi.ct = pp(ct, b); bi.q = pp(q, b); bi.u = pp(u, b); bi.g = pp(Gp, b); bi.b = pp(Bp, b); bi.qbuf = n * (size_t)p;
            bi.tr = tr;
            bi.tr.J = bshift_host(tr.J, (size_t)b * tr_slab); bi.tr.alpha = bshift_host(tr.alpha, (size_t)b * tr_slab);
            bi.tr.lambda = bshift_host(tr.lambda, (size_t)b * tr_slab); bi.tr.rule = bshift_host(tr.rule, (size_t)b * tr_slab);
            bi.tr.backtracks = bshift_host(tr.backtracks, (size_t)b * tr_slab);
            bi.b_is_array = b_is_array; bi.nchunks = (unsigned int)bt_chunks; bi.chunk_batches = (unsigned int)bt_batches;
            bi.part = pp(part_bt, b); bi.sync = pp(btsync, b);
            for (int j = 0; j < p; ++j) bi.bconst[j] = bconst_all[(size_t)b * kMaxP + j];
        }
        // all blocks in one strided copy
        SGP_CUDA_TRY(cudaMemcpy2DAsync(btinfo, slab ? slab : sizeof(BtInfo<T>), bis.data(), sizeof(BtInfo<T>), sizeof(BtInfo<T>), (size_t)nb, cudaMemcpyHostToDevice, st));
    }
    // ---- iteration loop
    if (any_running()) {
        int chunk = ro.check_every > 0 ? ro.check_every : (ro.stop_rule == SGP_STOP_MAXIT ? 200 : 20);
        if (algorithm == SGP_ALG_SGP && small_run) {
            // one launch runs every problem to its stopping rule (or to max_iter): the kernel tests the rules itself
            int done = 0;
            while (any_running()) {
                const int todo = ro.max_iter - done;
                if (todo < 1) { for (int b = 0; b < nb; ++b) if (status[b] == 0) status[b] = SGP_REASON_MAXIT; break; }
                if ((rc = launch_small(small_k, o, tr, bconst[0], todo, st))) return rc;
                if ((rc = read_ctrl())) return rc;
                done = ro.max_iter;
                for (int b = 0; b < nb; ++b) {
                    if (status[b] == 0) status[b] = hs[b].status;
                    if (status[b] == 0 && hs[b].k < done) done = hs[b].k;
                }
            }
        } else if (algorithm == SGP_ALG_SGP) {
            if (ro.max_iter == 0) { for (int b = 0; b < nb; ++b) if (status[b] == 0) status[b] = SGP_REASON_MAXIT; }
            else if ((rc = enqueue_ratio(Pb, 3, st))) return rc;        // K1 of iteration 0; every iteration enqueues the next one's
            int done = 0;
            while (any_running()) {
                int todo = ro.max_iter - done; if (todo > chunk) todo = chunk;
                if (todo < 1) { for (int b = 0; b < nb; ++b) if (status[b] == 0) status[b] = SGP_REASON_MAXIT; break; }
                if ((rc = enqueue_many(algorithm, todo, Pb, o, tr, bconst, b_is_array, st))) return rc;
                if ((rc = read_ctrl())) return rc;
                done = ro.max_iter;
                for (int b = 0; b < nb; ++b) {
                    if (status[b] == 0) status[b] = hs[b].status;
                    if (status[b] == 0 && hs[b].k < done) done = hs[b].k;      // the slowest problem still running
                }
            }
        } else if (algorithm == SGP_ALG_OSEM) {
            // max_iter cycles, then J0 (Eq.12) at the final iterate: q_j = A_j f for all j, as in the start-point phase
            int done = 0;
            if (rl_fused && ro.max_iter > 0) {     // row transform of h(0); every sub-step leaves the one of its result
                RowParams<T> P = Pb; P.in0 = f; P.maskmode = MM_NONE;
                if ((rc = launch_row(k_rowf[RF_PLAIN], P, 1, st))) return rc;
            }
            while (any_running() && done < ro.max_iter) {
                int todo = ro.max_iter - done; if (todo > chunk) todo = chunk;
                if ((rc = enqueue_many(algorithm, todo, Pb, o, tr, bconst, b_is_array, st))) return rc;
                done += todo;
                if ((rc = read_ctrl())) return rc;
                for (int b = 0; b < nb; ++b) if (status[b] == 0) status[b] = hs[b].status;
            }
            // Eq.25 stop (OSEM runs are never batched): the cycle counter and the error come from the device; the kernels of
            // the J0 phase test the device status, so it is cleared for them and the reason kept on the host
            const bool minerr_stop = status[0] == SGP_REASON_MINERR;
            const int k_minerr = hs[0].k;
            const double err_minerr = hs[0].err;
            if (minerr_stop) SGP_CUDA_TRY(cudaMemsetAsync(&ct->status, 0, sizeof(int), st));
            if (any_running() || minerr_stop) {
                Trace t0 = tr; t0.J = nullptr;
                RowParams<T> Pj = Pb; Pj.tr = t0;
                { RowParams<T> P = Pj; P.in0 = f; if ((rc = launch_row(k_rowf[RF_PLAIN], P, 1, st))) return rc; }
                { ColParams<T> Q = col_params(); Q.check_status = 1; if ((rc = launch_col(k_mult_run, Q, st))) return rc; }
                { RowParams<T> P = Pj; P.submode = QJ_INIT; P.in0 = Gp; P.in2 = Bp; P.out0 = q; P.part = part_J;
                  if ((rc = launch_row(k_rowi[RI_QJ], P, p, st))) return rc; }
                if ((rc = read_ctrl())) return rc;
                for (int b = 0; b < nb; ++b) {
                    if (status[b] == 0 || (minerr_stop && hs[b].status < 0)) status[b] = hs[b].status;
                    hs[b].k = minerr_stop ? k_minerr : done;
                    if (minerr_stop) hs[b].err = err_minerr;
                    if (status[b] == 0) status[b] = SGP_REASON_MAXIT;
                }
            }
        } else if (small_rl) {
            // RL rounds inside the cluster kernel (small.cuh): one launch runs every problem to its stopping rule
            int rounds = 0;
            while (any_running()) {
                int todo = ro.max_iter + 1 - rounds; if (todo < 1) todo = 1;
                if ((rc = launch_small(small_k_rl, o, tr, bconst[0], todo, st))) return rc;
                rounds += todo;
                if ((rc = read_ctrl())) return rc;
                for (int b = 0; b < nb; ++b) if (status[b] == 0) status[b] = hs[b].status;
            }
        } else {
            int rounds = 0;     // round k evaluates J0(f(k)) and, unless a rule fires, makes update k+1
            if (rl_fused) {     // row transform of f(0); every round leaves the one of f(k+1)
                RowParams<T> P = Pb; P.in0 = f; P.maskmode = MM_NONE;
                if ((rc = launch_row(k_rowf[RF_PLAIN], P, 1, st))) return rc;
            }
            while (any_running()) {
                int todo = ro.max_iter + 1 - rounds; if (todo > chunk) todo = chunk; if (todo < 1) todo = 1;
                if ((rc = enqueue_many(algorithm, todo, Pb, o, tr, bconst, b_is_array, st))) return rc;
                rounds += todo;
                if ((rc = read_ctrl())) return rc;
                for (int b = 0; b < nb; ++b) if (status[b] == 0) status[b] = hs[b].status;
            }
        }
    }
    SGP_CUDA_TRY(cudaEventRecord(ev2, st));
    if (nb > 1) {
        final_update_batched_kernel<T><<<dim3(ew_grid(n), 1, nb), 256, 0, st>>>(tab, f, d, n, ct, slab);     // a10: the last accepted step, if still pending
        launches++;
    } else {
        final_update_kernel<T><<<ew_grid(n), 256, 0, st>>>(f, d, (T *)f_out[0], n, ct);
        launches++;
    }
    SGP_CUDA_TRY(cudaGetLastError());
    // traces: batched plans bring every trace array of all problems to the host in ONE strided copy and hand the rows out from there
    int kmax = 0;
    for (int b = 0; b < nb; ++b) if (hs[b].k > kmax) kmax = hs[b].k;
    struct TraceCopy { void *dev; size_t elem; int extra; bool any; std::vector<unsigned char> host; };
    TraceCopy tcs[6] = {{trJ, sizeof(double), 1, false, {}}, {tr.err ? trE : nullptr, sizeof(double), 2, false, {}}, {trA, sizeof(double), 0, false, {}},
                        {trL, sizeof(double), 0, false, {}}, {trR, sizeof(int), 0, false, {}}, {trB, sizeof(int), 0, false, {}}};
    auto wanted = [&](const sgp_result &R, int i) -> void * {
        switch (i) { case 0: return R.trace_J; case 1: return R.trace_err; case 2: return R.trace_alpha; case 3: return R.trace_lambda;
                     case 4: return R.trace_rule; default: return R.trace_backtracks; }
    };
    if (nb > 1) {
        for (int i = 0; i < 6; ++i) {
            TraceCopy &t = tcs[i];
            if (!t.dev) continue;
            for (int b = 0; b < nb; ++b) if (wanted(res[b], i) && hs[b].k + t.extra > 0) t.any = true;
            if (!t.any) continue;
            const size_t width = t.elem * (size_t)(kmax + t.extra);
            t.host.resize(width * (size_t)nb);
            SGP_CUDA_TRY(cudaMemcpy2DAsync(t.host.data(), width, t.dev, tr_slab, width, (size_t)nb, cudaMemcpyDeviceToHost, st));
        }
    } else {
        const int b = 0;
        const int kdone = hs[b].k;
        const size_t to = (size_t)b * tr_slab;
        sgp_result &R = res[b];
        if (R.trace_J) SGP_CUDA_TRY(cudaMemcpyAsync(R.trace_J, bshift_host(trJ, to), sizeof(double) * (kdone + 1), cudaMemcpyDeviceToHost, st));
        if (R.trace_err && tr.err) SGP_CUDA_TRY(cudaMemcpyAsync(R.trace_err, bshift_host(trE, to), sizeof(double) * (kdone + 2), cudaMemcpyDeviceToHost, st));
        if (kdone > 0) {
            if (R.trace_alpha) SGP_CUDA_TRY(cudaMemcpyAsync(R.trace_alpha, bshift_host(trA, to), sizeof(double) * kdone, cudaMemcpyDeviceToHost, st));
            if (R.trace_lambda) SGP_CUDA_TRY(cudaMemcpyAsync(R.trace_lambda, bshift_host(trL, to), sizeof(double) * kdone, cudaMemcpyDeviceToHost, st));
            if (R.trace_rule) SGP_CUDA_TRY(cudaMemcpyAsync(R.trace_rule, bshift_host(trR, to), sizeof(int) * kdone, cudaMemcpyDeviceToHost, st));
            if (R.trace_backtracks) SGP_CUDA_TRY(cudaMemcpyAsync(R.trace_backtracks, bshift_host(trB, to), sizeof(int) * kdone, cudaMemcpyDeviceToHost, st));
        }
    }
    SGP_CUDA_TRY(cudaStreamSynchronize(st));
    if (nb > 1) {
        for (int i = 0; i < 6; ++i) {
            const TraceCopy &t = tcs[i];
            if (!t.any) continue;
            const size_t width = t.elem * (size_t)(kmax + t.extra);
            for (int b = 0; b < nb; ++b) {
                void *dst = wanted(res[b], i);
                const int cnt = hs[b].k + t.extra;
                if (dst && cnt > 0) memcpy(dst, t.host.data() + (size_t)b * width, t.elem * (size_t)cnt);
            }
        }
    }
    if (profiling) prof_collect();
    float ms01 = 0.f, ms12 = 0.f;
    cudaEventElapsedTime(&ms01, ev0, ev1);
    cudaEventElapsedTime(&ms12, ev1, ev2);
    int worst = SGP_OK;
    for (int b = 0; b < nb; ++b) {
        const Ctrl &h = hs[b];
        sgp_result &R = res[b];
        R.iterations = h.k;
        R.stop_reason = status[b] > 0 ? status[b] : 0;
        R.J0_final = h.J;
        R.discrepancy_final = 2.0 * h.J / o.nS_total;
        R.total_backtracks = h.total_backtracks;
        R.L1_used = algorithm == SGP_ALG_SGP ? h.L1 : 0.0;
        R.L2_used = algorithm == SGP_ALG_SGP ? h.L2 : 0.0;
        R.n_fft2 = (long)(h.nfft - nfft0[b]);
        R.err_final = tr.err ? h.err : 0.0;
        R.setup_ms = ms01; R.loop_ms = ms12;
        R.kernel_launches = launches - launches0;
        R.fused_linesearch = ((algorithm == SGP_ALG_SGP && small_run) || small_rl) ? 2 : (algorithm == SGP_ALG_SGP && fuse_ls) ? 1 : 0;
        R.status = status[b] < 0 ? status[b] : SGP_OK;
        if (status[b] < 0 && worst == SGP_OK) worst = status[b];
    }
    return worst;
}

PlanBase *SGP_MAKE() { return new PlanImpl<SGP_T>(); }

}  // namespace sgpk
