// plan_impl.inl -- included by plan_f32.cu / plan_f64.cu with SGP_T and SGP_MAKE defined.
#include "plan.cuh"
#include "small_params.h"

namespace sgpk {

template <typename T> struct PlanImpl : PlanBase {
    using C = cx<T>;
    size_t n = 0, nspec = 0;       // reals per plane, complex numbers per half spectrum (= n/2)
    int lnb = 1;                   // problems per launch: nb inside run_batched, 1 in the set-up paths (which work on shared buffers)
    size_t slab = 0, tr_slab = 0;  // batched plans: bytes between the per-problem arrays / the trace blocks of consecutive problems
    int Lr = 0, Lc = 0;            // FFT lengths: nx/2 (rows), ny (columns)
    bool use_pdl = true;
    bool fuse_ls = true;           // line-search kernel fused with the next iteration's ratio + row FFT (row_inv RI_LSF)
    int row_threads = 0, col_threads = 0, nrb = 0, ntiles = 0, nsm = 0, col_grid = 0;
    size_t bt_chunks = 0, bt_batches = 1;   // chunks per Armijo trial and batches per chunk (aux.cuh: backtrack_rounds)
    size_t row_smem = 0, col_smem = 0;
    row_kernel_t<T> k_rowf[RF_NMODES] = {nullptr}, k_rowi[RI_NMODES] = {nullptr};
    col_kernel_t<T> k_colf = nullptr, k_conj = nullptr, k_mult = nullptr;
    col_kernel_t<T> k_conj1 = nullptr, k_mult1 = nullptr;
    bool col2 = false;             // single-image product kernels also exist in their two-CTAs-per-SM form (col2_kernel)
    col_kernel_t<T> k_conj2 = nullptr, k_mult2 = nullptr;
    col_kernel_t<T> k_conj_run = nullptr, k_mult_run = nullptr;   // the pair the current run uses
    int col2_threads = 0; size_t col2_smem = 0;
    C *tw_c2 = nullptr;            // pass tables of the 32-elements-per-thread column plan      // single-image forms (OSEM sub-steps, A_j / A_j^T alone)
    // device memory
    std::vector<void *> allocs;
    C *tw_r = nullptr, *tw_h = nullptr, *tw_c = nullptr, *pack = nullptr;
    C *khat = nullptr, *khatB = nullptr, *spec = nullptr;
    T *Gp = nullptr, *Bp = nullptr, *q = nullptr, *u = nullptr, *f = nullptr, *grad = nullptr, *d = nullptr;
    T *alphaR = nullptr, *alpha = nullptr, *scratch = nullptr;
    T *alphaJ = nullptr;           // boundary problems: alpha_j on R, 0 elsewhere, p planes (OSEM, Eq.22)
    unsigned char *MR = nullptr;
    double *part_bb = nullptr, *part_gd = nullptr, *part_J = nullptr, *part_bt = nullptr, *part_misc = nullptr;
    Ctrl *ct = nullptr;
    BtInfo<T> *btinfo = nullptr;
    unsigned int *btsync = nullptr, *fxsync = nullptr;
    Ctrl *ct_shadow = nullptr;      // refresh round (A21): control block whose status tells the column pass whether this is a refresh iteration
    double *part_fx = nullptr, *part_err = nullptr;
    size_t fx_chunks = 0, fx_batches = 1;
    C *khatB_tmp = nullptr;        // companion line of the Gaussian's transfer function (smoothed constant start)
    small_kernel_t<T> small_k = nullptr;   // small grids: the whole SGP iteration in one kernel, one cluster per problem (small.cuh)
    small_kernel_t<T> small_k_rl = nullptr; // the same for Richardson-Lucy rounds
    int small_nc = 0, small_threads = 0, small_er = 0, small_ec = 0; size_t small_smem = 0;
    C *tw_sr = nullptr, *tw_sc = nullptr;   // pass tables of its row / column FFT plans
    const void **ptrtab = nullptr;  // batched plans: addresses of the caller's arrays of a run (aux.cuh: BatchTab), 2 nb p + 2 nb entries
    // per-run trace buffers
    double *trJ = nullptr, *trA = nullptr, *trL = nullptr, *fA = nullptr, *fL = nullptr, *trE = nullptr;
    int *trR = nullptr, *trB = nullptr;
    int trace_cap = 0;
    cudaEvent_t ev0 = nullptr, ev1 = nullptr, ev2 = nullptr;
    cudaStream_t cap_stream = nullptr;       // stream the iteration graph is captured on (use_graph)
    cudaGraphExec_t gexec = nullptr;         // kept across run() calls, re-captured when gsig changes
    struct GraphSig {                        // everything the captured launches carry by value
        int algorithm, b_is_array; DevOpts o; Trace tr; double bconst[kMaxP];
        bool fuse_ls, rl_fused; const void *k_conj, *k_mult, *truth;
    } gsig;
    const void *run_truth = nullptr;         // Eq.25: the true object of the current run (device pointer)
    bool run_graph = true;                   // this run replays graphs (per-run use_graph bit 0)
    bool rl_fused = true;                    // RL / OSEM on the four-launch schedule, else six launches
    long graph_launches = 0;                 // kernels in one replay of gexec
    // per-kernel timing (sgp_plan_set_profiling): one event pair per launch of the iteration loop
    struct ProfRec { int slot; cudaEvent_t a, b; };
    std::vector<ProfRec> prof_recs;
    std::vector<cudaEvent_t> prof_pool;
    size_t prof_used = 0;
    int cur_slot = -1;

    ~PlanImpl() override
    {
        for (void *a : allocs) cudaFree(a);
        free_trace();
        if (ev0) cudaEventDestroy(ev0);
        if (ev1) cudaEventDestroy(ev1);
        if (ev2) cudaEventDestroy(ev2);
        if (gexec) cudaGraphExecDestroy(gexec);
        if (cap_stream) cudaStreamDestroy(cap_stream);
        for (cudaEvent_t e : prof_pool) cudaEventDestroy(e);
    }
    cudaEvent_t prof_event()
    {
        if (prof_used == prof_pool.size()) {
            cudaEvent_t e = nullptr;
            if (cudaEventCreate(&e) != cudaSuccess) return nullptr;
            prof_pool.push_back(e);
        }
        return prof_pool[prof_used++];
    }
    // bracket the next launch with events when profiling is on and a slot is selected
    struct ProfScope {
        PlanImpl *P; cudaStream_t st; cudaEvent_t a = nullptr;
        ProfScope(PlanImpl *P_, cudaStream_t st_) : P(P_), st(st_)
        {
            if (P->profiling && P->cur_slot >= 0 && (a = P->prof_event())) cudaEventRecord(a, st);
        }
        ~ProfScope()
        {
            if (a) { cudaEvent_t b = P->prof_event(); if (b) { cudaEventRecord(b, st); P->prof_recs.push_back({P->cur_slot, a, b}); } }
        }
    };
    void prof_reset() { prof_recs.clear(); prof_used = 0; for (int i = 0; i < SGP_PROF_SLOTS; ++i) { prof_ms[i] = 0.0; prof_count[i] = 0; } }
    void prof_collect()
    {
        for (const ProfRec &r : prof_recs) {
            float ms = 0.f;
            if (cudaEventElapsedTime(&ms, r.a, r.b) == cudaSuccess) { prof_ms[r.slot] += ms; prof_count[r.slot]++; }
        }
        prof_recs.clear(); prof_used = 0;
    }
    void free_trace()
    {
        cudaFree(trJ);      // one block: trJ, trA, trL, fA, fL, trR, trB
        trJ = trA = trL = fA = fL = trE = nullptr; trR = trB = nullptr; trace_cap = 0;
    }
    // The workspace is ONE device allocation (a cudaMalloc / cudaFree pair costs ~0.5 ms and synchronises the device:
    // two dozen of them were a third of a one-shot call): dalloc() only records a request, commit_allocs() allocates
    // the arena, hands out 256-byte aligned pieces and performs the deferred table uploads.
    struct Req { void **ptr; size_t bytes; };
    struct Upload { void **ptr; std::vector<unsigned char> data; };
    std::vector<Req> reqs;
    std::vector<Upload> uploads;
    template <typename U> int dalloc(U **ptr, size_t count)
    {
        reqs.push_back({reinterpret_cast<void **>(ptr), count * sizeof(U)});
        return SGP_OK;
    }
    // per-problem arrays: one slab per problem (nb of them, identical layout); *ptr is problem 0's copy
    std::vector<Req> reqs_pp;
    template <typename U> int dalloc_pp(U **ptr, size_t count)
    {
        // an ordinary plan keeps everything in ONE arena, in the order of the requests: the column passes stream a spectrum
        // tile and the transfer-function tile of the same offset at once, and how far apart the two planes lie decides how
        // the two streams share the L2 slices (measured: with the spectra in an allocation of their own K2 / K5 took
        // 45 / 45 us instead of 39 / 37 us at 3 x 2048^2)
        if (nb == 1) return dalloc(ptr, count);
        reqs_pp.push_back({reinterpret_cast<void **>(ptr), count * sizeof(U)});
        return SGP_OK;
    }
    template <typename U> static U *bshift_host(U *ptr, size_t off)
    {
        return ptr ? reinterpret_cast<U *>(reinterpret_cast<unsigned char *>(const_cast<typename std::remove_const<U>::type *>(ptr)) + off) : ptr;
    }
    // pieces of 64 KB and more start on a 4 KB boundary (the 64 KB tiles of spectra and transfer functions are moved by bulk
    // copies: with the planes on odd multiples of 256 bytes the column passes of 3 x 2048^2 took 45 us instead of 39 us), the
    // small ones on 256 bytes
    static size_t piece_align(size_t bytes) { return bytes >= 65536 ? 4096 : 256; }
    static size_t place(size_t &off, size_t bytes)
    {
        const size_t a = piece_align(bytes);
        off = (off + a - 1) & ~(a - 1);
        const size_t at = off;
        off += bytes;
        return at;
    }
    int commit_allocs()
    {
        size_t total = 0;
        for (const Req &r : reqs) place(total, r.bytes);
        total = (total + 4095) & ~(size_t)4095;
        void *raw = nullptr;
        SGP_CUDA_TRY(cudaMalloc(&raw, total ? total : 256));
        allocs.push_back(raw);
        bytes_allocated += total;
        size_t off = 0;
        for (const Req &r : reqs) { const size_t at = place(off, r.bytes); *r.ptr = static_cast<unsigned char *>(raw) + at; }
        reqs.clear();
        size_t per = 0;
        for (const Req &r : reqs_pp) place(per, r.bytes);
        per = (per + 4095) & ~(size_t)4095;
        void *raw_pp = nullptr;
        SGP_CUDA_TRY(cudaMalloc(&raw_pp, per * (size_t)nb ? per * (size_t)nb : 256));
        allocs.push_back(raw_pp);
        bytes_allocated += per * (size_t)nb;
        off = 0;
        for (const Req &r : reqs_pp) { const size_t at = place(off, r.bytes); *r.ptr = static_cast<unsigned char *>(raw_pp) + at; }
        reqs_pp.clear();
        slab = nb > 1 ? per : 0;
        for (const Upload &u : uploads) SGP_CUDA_TRY(cudaMemcpy(*u.ptr, u.data.data(), u.data.size(), cudaMemcpyHostToDevice));
        uploads.clear();
        return SGP_OK;
    }

    int init() override
    {
        n = (size_t)ny * nx; nspec = n / 2;
        use_pdl = getenv("SGP_PDL") != nullptr;      // measured: no gain on B200 at 2048^2 (profiles/), off by default
        Lr = nx / 2; Lc = ny;
        constexpr int dummy = 0; (void)dummy;
        const int Er = fft_E<T>(Lr), Ec = fft_E_col<T>(Lc);
        for (int m = 0; m < RF_NMODES; ++m) if (!(k_rowf[m] = get_row_fwd<T>(Lr, m, G.masked != 0))) return SGP_ERR_ARG;
        for (int m = 0; m < RI_NMODES; ++m) if (!(k_rowi[m] = get_row_inv<T>(Lr, m, G.masked != 0))) return SGP_ERR_ARG;
        int Cc = 0, RB = 0;
        int rc = choose_tiles(ny, nx, dtype, &opt, &Cc, &RB, nb);
        if (rc) return rc;
        const bool multi = p > 1;
        // batched plans (nb > 1) use the column kernels compiled with the per-problem offset (col.cuh: BATCH), asked for by a negative width
        const int Cq = nb > 1 ? -Cc : Cc;
        k_colf = get_col<T>(Lc, CM_FWD, false); k_conj = get_col<T>(Lc, CM_CONJSUM, multi, Cq); k_mult = get_col<T>(Lc, CM_MULT, multi, Cq);
        k_conj1 = get_col<T>(Lc, CM_CONJSUM, false, Cq); k_mult1 = get_col<T>(Lc, CM_MULT, false, Cq);
        if (!k_colf || !k_conj || !k_mult || !k_conj1 || !k_mult1) return SGP_ERR_ARG;
        G.C = Cc; G.RB = RB; G.lc = 0; while ((1 << G.lc) < Cc) G.lc++;
        row_threads = RB * group_threads(Lr / Er);
        col_threads = Cc * (Lc / Ec);
        nrb = ny / RB; ntiles = Lr / Cc;
        row_smem = ((size_t)RB * row_stride(Lr, Er) + row_table_entries<T>(Lr)) * sizeof(C);     // rows + twiddle tables (row_fwd.cuh)
        col_smem = ((size_t)Cc * fft_padded_len(Lc, Ec) + 2 * (size_t)Cc * Lc) * sizeof(C);
        if (row_threads > 256 || col_threads > 512 || row_smem > 227 * 1024 || col_smem > 227 * 1024) return SGP_ERR_ARG;
        for (int m = 0; m < RF_NMODES; ++m)
            SGP_CUDA_TRY(cudaFuncSetAttribute((const void *)k_rowf[m], cudaFuncAttributeMaxDynamicSharedMemorySize, (int)row_smem));
        for (int m = 0; m < RI_NMODES; ++m)
            SGP_CUDA_TRY(cudaFuncSetAttribute((const void *)k_rowi[m], cudaFuncAttributeMaxDynamicSharedMemorySize, (int)row_smem));
        SGP_CUDA_TRY(cudaFuncSetAttribute((const void *)k_colf, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)col_smem));
        SGP_CUDA_TRY(cudaFuncSetAttribute((const void *)k_conj, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)col_smem));
        SGP_CUDA_TRY(cudaFuncSetAttribute((const void *)k_mult, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)col_smem));
        SGP_CUDA_TRY(cudaFuncSetAttribute((const void *)k_conj1, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)col_smem));
        SGP_CUDA_TRY(cudaFuncSetAttribute((const void *)k_mult1, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)col_smem));
        int dev = 0;
        SGP_CUDA_TRY(cudaGetDevice(&dev));
        SGP_CUDA_TRY(cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev));
        // Fused or separate line-search / ratio kernels.  Round 1 chose by the size of the hand-off (g_j, q_j, u_j: 3p planes) against
        // L2 and ran 2048^2 single image separate; with the backtracking folded into the ratio kernel (six launches instead of
        // seven) the fused form is ahead there too (112.7 vs 113.2 us per iteration; 3 x 2048^2: 209 vs 222 us), so it is the default.
        fuse_ls = true;
        if (opt.use_graph & 4) fuse_ls = false;      // experiment switches
        if (opt.use_graph & 8) fuse_ls = true;
        col_grid = (opt.use_graph & 2) ? (ntiles < nsm ? ntiles : nsm) : ntiles;   // experiment switch: persistent or one tile per CTA

        // Small grids: one image (with or without boundary-effect correction) at 128^2 / 256^2 iterates inside ONE kernel run by
        // one thread-block cluster per problem (small.cuh) when the device can co-schedule such a cluster; use_graph bit 7 (or any other
        // experiment switch) keeps the launch-per-pass path.  Batched plans run one cluster per problem: the device holds 7 clusters of 16 CTAs
        // in the one-CTA-per-SM form of the kernel and 14 in its two-CTAs-per-SM form, which is taken when the batch is larger than 7.
        // Aggregate kit/s at 256^2, 100 iterations per problem (form 1 / form 2 / launch-per-pass): 4 problems 163 / 154 / 71, 8 problems
        // 177 / 230 / 121, 16 problems 230 / 272 / 195, 32 problems 281 / 346 / 326, 64 problems 292 / 385 / 396 -- so 256^2 batches of more
        // than 32 problems stay launch-per-pass; 128^2 (clusters of 8) always runs in clusters.
        if (p == 1 && (opt.use_graph & ~1) == 0 && !getenv("SGP_NO_CLUSTER")) {      // any experiment switch: launch-per-pass
            // which form: one CTA per SM (255 registers, planes prefetched) while the device holds all clusters of the plan at once,
            // two CTAs per SM for larger batches; SGP_SMALL_FORM = 1 / 2 forces one (experiments)
            auto max_clusters = [&](small_kernel_t<T> kk) -> int {
                if (!kk) return 0;
                bool ok = cudaFuncSetAttribute((const void *)kk, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)small_smem) == cudaSuccess;
                if (ok && small_nc > 8) ok = cudaFuncSetAttribute((const void *)kk, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) == cudaSuccess;
                int nclusters = 0;
                if (ok) {
                    cudaLaunchConfig_t cfg;
                    memset(&cfg, 0, sizeof(cfg));
                    cfg.gridDim = dim3(small_nc); cfg.blockDim = dim3(small_threads); cfg.dynamicSmemBytes = small_smem;
                    cudaLaunchAttribute at[1];
                    at[0].id = cudaLaunchAttributeClusterDimension;
                    at[0].val.clusterDim.x = small_nc; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
                    cfg.attrs = at; cfg.numAttrs = 1;
                    ok = cudaOccupancyMaxActiveClusters(&nclusters, (const void *)kk, &cfg) == cudaSuccess;
                }
                if (!ok) { (void)cudaGetLastError(); return 0; }
                return nclusters;
            };
            small_kernel_t<T> k1 = get_small<T>(ny, nx, G.masked != 0, false, false, &small_nc, &small_threads, &small_smem, &small_er, &small_ec);
            const int c1 = max_clusters(k1);
            bool two = false;
            if (k1 && nb > c1) {     // only where the second form really holds more clusters (at 128^2 the first already has two CTAs per SM)
                int a_, b_, e_, f_; size_t c_;
                two = max_clusters(get_small<T>(ny, nx, G.masked != 0, false, true, &a_, &b_, &c_, &e_, &f_)) > c1;
            }
            if (const char *f = getenv("SGP_SMALL_FORM")) two = f[0] == '2';
            small_k = get_small<T>(ny, nx, G.masked != 0, false, two, &small_nc, &small_threads, &small_smem, &small_er, &small_ec);
            small_k_rl = small_k ? get_small<T>(ny, nx, G.masked != 0, true, two, &small_nc, &small_threads, &small_smem, &small_er, &small_ec) : nullptr;
            const int cs = max_clusters(small_k), cr = max_clusters(small_k_rl);
            if (getenv("SGP_SMALL_DEBUG")) fprintf(stderr, "[sgp] cluster kernel: nb %d, clusters resident: form 1 %d, chosen form %d: %d (RL %d)\n", nb, c1, two ? 2 : 1, cs, cr);
            if (cs < 1) small_k = nullptr;
            if (cr < 1) small_k_rl = nullptr;
            if (small_k && nb > 32 && small_nc > 8 && !getenv("SGP_SMALL_FORM")) { small_k = nullptr; small_k_rl = nullptr; }
            if (!small_k) small_k_rl = nullptr;
        }
        // twiddles, computed in double on the host
        std::vector<C> h;
        auto upload = [&](C **dst, int len, int count) -> int {     // exp(-2 pi i k / len), k < count
            h.resize(count);
            for (int k = 0; k < count; ++k) {
                double a = -2.0 * M_PI * (double)k / (double)len;
                h[k].x = (T)cos(a); h[k].y = (T)sin(a);
            }
            int r = dalloc(dst, (size_t)count + 2);      // + padding: the kernels copy the tables in 16-byte pieces
            if (r) return r;
            const unsigned char *b = reinterpret_cast<const unsigned char *>(h.data());
            uploads.push_back({reinterpret_cast<void **>(dst), std::vector<unsigned char>(b, b + sizeof(C) * count)});
            return SGP_OK;
        };
        auto upload_passes = [&](C **dst, int Lf, int Ef) -> int {  // per-pass tables [r-1][j mod NS] (fft_core.cuh)
            h.assign((size_t)tw_total(Lf, Ef), C{(T)1, (T)0});
            for (int ip = 1; plan_radix(Lf, Ef, ip) != 0; ++ip) {
                const int R = plan_radix(Lf, Ef, ip), NS = plan_ns(Lf, Ef, ip), off = tw_offset(Lf, Ef, ip);
                for (int r = 1; r < R; ++r)
                    for (int jm = 0; jm < NS; ++jm) {
                        double a = -2.0 * M_PI * (double)r * (double)jm / ((double)NS * (double)R);
                        h[off + (r - 1) * NS + jm].x = (T)cos(a); h[off + (r - 1) * NS + jm].y = (T)sin(a);
                    }
            }
            int r = dalloc(dst, h.size() + 2);
            if (r) return r;
            const unsigned char *b = reinterpret_cast<const unsigned char *>(h.data());
            uploads.push_back({reinterpret_cast<void **>(dst), std::vector<unsigned char>(b, b + sizeof(C) * h.size())});
            return SGP_OK;
        };
        if ((rc = upload_passes(&tw_r, Lr, Er))) return rc;
        if ((rc = upload(&tw_h, nx, Lr + 1))) return rc;
        if ((rc = upload_passes(&tw_c, Lc, Ec))) return rc;
        if (small_k) { if ((rc = upload_passes(&tw_sr, Lr, small_er))) return rc; if ((rc = upload_passes(&tw_sc, Lc, small_ec))) return rc; }
        // single-image product passes: the two-CTAs-per-SM kernel where it exists (float, 256 threads at this tile width);
        // run() decides per algorithm whether to use it
        k_conj_run = k_conj; k_mult_run = k_mult;
        if (p == 1 && nb == 1 && !(opt.use_graph & 16) && plan_ok(Lc, 32) && Cc * (Lc / 32) == 256) {
            col_kernel_t<T> c2 = get_col2<T>(Lc, CM_CONJSUM), m2 = get_col2<T>(Lc, CM_MULT);
            const size_t sm2 = (size_t)Cc * fft_padded_len(Lc, 32) * sizeof(C);
            if (c2 && m2 && sm2 <= 113 * 1024) {
                SGP_CUDA_TRY(cudaFuncSetAttribute((const void *)c2, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm2));
                SGP_CUDA_TRY(cudaFuncSetAttribute((const void *)m2, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm2));
                if ((rc = upload_passes(&tw_c2, Lc, 32))) return rc;
                k_conj2 = c2; k_mult2 = m2; col2 = true; col2_threads = 256; col2_smem = sm2;
            }
        }
        if ((rc = dalloc_pp(&pack, (size_t)ny))) return rc;
        if ((rc = dalloc(&khat, nspec * p))) return rc;
        if ((rc = dalloc(&khatB, (size_t)ny * p))) return rc;
        if ((rc = dalloc_pp(&spec, nspec * p))) return rc;
        if ((rc = dalloc_pp(&Gp, n * p))) return rc;
        if ((rc = dalloc_pp(&Bp, n * p))) return rc;
        if ((rc = dalloc_pp(&q, 2 * n * p))) return rc;          // double-buffered (Ctrl::qsel)
        if ((rc = dalloc_pp(&u, n * p))) return rc;
        if ((rc = dalloc_pp(&f, n))) return rc;
        if ((rc = dalloc_pp(&grad, n))) return rc;
        if ((rc = dalloc_pp(&d, n))) return rc;
        if ((rc = dalloc(&scratch, n))) return rc;
        if (G.masked) {
            if ((rc = dalloc(&alphaR, n))) return rc;
            if ((rc = dalloc(&alpha, n))) return rc;
            if ((rc = dalloc(&MR, n))) return rc;
            if ((rc = dalloc(&alphaJ, n * p))) return rc;
        }
        if ((rc = dalloc_pp(&part_bb, (size_t)nrb * 4))) return rc;
        if ((rc = dalloc_pp(&part_gd, (size_t)nrb))) return rc;
        if ((rc = dalloc_pp(&part_J, (size_t)nrb * p * 2))) return rc;
        {   // one chunk per CTA of the ratio kernel (grid nrb x p), in whole batches
            const size_t batch = bt_chunk_elems<T>(), total = (size_t)p * n, ctas = (size_t)nrb * p;
            bt_batches = (total + batch * ctas - 1) / (batch * ctas);
            if (bt_batches < 1) bt_batches = 1;
            bt_chunks = (total + batch * bt_batches - 1) / (batch * bt_batches);
        }
        if ((rc = dalloc_pp(&part_bt, bt_chunks))) return rc;
        if ((rc = dalloc_pp(&part_misc, (size_t)1024 * p))) return rc;
        if ((rc = dalloc_pp(&ct, (size_t)1))) return rc;
        if ((rc = dalloc_pp(&btinfo, (size_t)1))) return rc;
        if ((rc = dalloc_pp(&btsync, (size_t)kBtSyncWords))) return rc;
        if ((rc = dalloc(&fxsync, (size_t)kBtSyncWords))) return rc;
        if ((rc = dalloc(&ct_shadow, (size_t)1))) return rc;
        {   // flux-constrained projection (extra.cuh): about two chunks per SM and Newton step
            const size_t batch = bt_chunk_elems<T>(), ctas = 2 * (size_t)nsm;
            fx_batches = (n + batch * ctas - 1) / (batch * ctas);
            if (fx_batches < 1) fx_batches = 1;
            fx_chunks = (n + batch * fx_batches - 1) / (batch * fx_batches);
        }
        if ((rc = dalloc(&part_fx, 3 * fx_chunks))) return rc;
        if ((rc = dalloc(&part_err, (size_t)2 * 1184))) return rc;
        if ((rc = dalloc(&khatB_tmp, (size_t)ny))) return rc;
        if (nb > 1 && (rc = dalloc(&ptrtab, (size_t)2 * nb * p + 2 * (size_t)nb))) return rc;
        if ((rc = commit_allocs())) return rc;
        for (int b = 0; b < nb; ++b) SGP_CUDA_TRY(cudaMemset(bshift_host(ct, (size_t)b * slab), 0, sizeof(Ctrl)));
        SGP_CUDA_TRY(cudaEventCreate(&ev0));
        SGP_CUDA_TRY(cudaEventCreate(&ev1));
        SGP_CUDA_TRY(cudaEventCreate(&ev2));
        return SGP_OK;
    }

    // ------------------------------------------------------------------ launch helpers
    RowParams<T> row_params() const
    {
        RowParams<T> P;
        memset(&P, 0, sizeof(P));
        P.G = G; P.ct = ct;
        P.plane = n; P.specplane = nspec; P.spec = spec; P.qbuf = n * (size_t)p;
        P.tw = tw_r; P.twh = tw_h; P.alphaR = alphaR; P.slab = lnb > 1 ? slab : 0; P.tr_slab = lnb > 1 ? tr_slab : 0;
        return P;
    }
    // launch with programmatic stream serialisation: the kernel may be scheduled while its predecessor drains and
    // waits for it in pdl_wait() (ew.cuh)
    template <typename K, typename PT>
    int launch_pdl(K k, dim3 grid, int threads, size_t smem, const PT &P, cudaStream_t st)
    {
        ProfScope ps(this, st);
        cudaLaunchConfig_t cfg;
        memset(&cfg, 0, sizeof(cfg));
        cfg.gridDim = grid; cfg.blockDim = dim3(threads); cfg.dynamicSmemBytes = smem; cfg.stream = st;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        at[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = at; cfg.numAttrs = use_pdl ? 1 : 0;
        SGP_CUDA_TRY(cudaLaunchKernelEx(&cfg, k, P));
        launches++;
        return SGP_OK;
    }
    int launch_row(row_kernel_t<T> k, const RowParams<T> &P, int images, cudaStream_t st)
    {
        return launch_pdl(k, dim3(nrb, images, lnb), row_threads, row_smem, P, st);
    }
    ColParams<T> col_params() const
    {
        ColParams<T> P;
        memset(&P, 0, sizeof(P));
        P.G = G; P.ct = ct; P.in = spec; P.out = spec; P.khat = khat; P.khatB = khatB;
        P.specplane = nspec; P.tw = tw_c; P.pack = pack; P.p = p; P.ntiles = ntiles; P.slab = lnb > 1 ? slab : 0;
        P.pf_ahead = (col_grid == ntiles && ntiles > nsm && lnb == 1) ? nsm : 0;      // col.cuh: SGP_COL_PF2
        return P;
    }
    int launch_col(col_kernel_t<T> k, const ColParams<T> &P, cudaStream_t st)
    {
        if (col2 && (k == k_conj2 || k == k_mult2)) {     // one tile per CTA, its own pass tables
            ColParams<T> Q = P; Q.tw = tw_c2;
            return launch_pdl(k, dim3(ntiles, 1, lnb), col2_threads, col2_smem, Q, st);
        }
        return launch_pdl(k, dim3(col_grid, 1, lnb), col_threads, col_smem, P, st);
    }
    // `iters` SGP iterations of all lnb problems in one launch, one cluster per problem (small.cuh)
    int launch_small(small_kernel_t<T> kern, const DevOpts &o, const Trace &tr, double bconst0, int iters, cudaStream_t st)
    {
        SmallParams<T> S;
        memset(&S, 0, sizeof(S));
        S.G = G; S.o = o; S.tr = tr; S.ct = ct; S.f = f; S.grad = grad; S.d = d; S.q = q; S.g = Gp; S.alphaR = alphaR; S.qbuf = n * (size_t)p;
        S.khat = khat; S.khatB = khatB; S.tw_r = tw_sr; S.tw_h = tw_h; S.tw_c = tw_sc; S.bconst = bconst0; S.iters = iters;
        S.slab = lnb > 1 ? slab : 0; S.tr_slab = lnb > 1 ? tr_slab : 0;
        cudaLaunchConfig_t cfg;
        memset(&cfg, 0, sizeof(cfg));
        cfg.gridDim = dim3(small_nc * lnb); cfg.blockDim = dim3(small_threads); cfg.dynamicSmemBytes = small_smem; cfg.stream = st;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.x = small_nc; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
        cfg.attrs = at; cfg.numAttrs = 1;
#ifdef SGP_SMALL_TIMING
        static unsigned long long *dbg = nullptr;
        if (!dbg) cudaMalloc(&dbg, 64 * sizeof(unsigned long long));
        cudaMemsetAsync(dbg, 0, 64 * sizeof(unsigned long long), st);
        S.dbg = dbg;
#endif
        SGP_CUDA_TRY(cudaLaunchKernelEx(&cfg, kern, S));
        launches++;
#ifdef SGP_SMALL_TIMING
        if (getenv("SGP_SMALL_DBG")) {
            unsigned long long h[64];
            cudaStreamSynchronize(st);
            cudaMemcpy(h, dbg, sizeof(h), cudaMemcpyDeviceToHost);
            fprintf(stderr, "[small timing, ns]");
            for (int i = 1; i < 64 && h[i]; ++i) fprintf(stderr, " %llu", h[i] - h[i - 1]);
            fprintf(stderr, "\n");
        }
#endif
        return SGP_OK;
    }
    static int ew_grid(size_t count) { size_t b = (count + 255) / 256; return (int)(b > 1184 ? 1184 : (b < 1 ? 1 : b)); }

    // ------------------------------------------------------------------ transfer functions and boundary weights
    int set_psf(const void *const *psf, cudaStream_t st) override
    {
        if (!psf) return SGP_ERR_ARG;
        for (int j = 0; j < p; ++j) if (!psf[j]) return SGP_ERR_ARG;
        const int cy = opt.psf_origin == SGP_PSF_CENTER ? ny / 2 : 0, cxs = opt.psf_origin == SGP_PSF_CENTER ? nx / 2 : 0;
        int rc;
        for (int j = 0; j < p; ++j) {
            plane_sum_kernel<T><<<ew_grid(n), 256, 0, st>>>((const T *)psf[j], n, ct, part_err);
            launches++;
            Ctrl h;
            SGP_CUDA_TRY(cudaMemcpyAsync(&h, ct, sizeof(Ctrl), cudaMemcpyDeviceToHost, st));
            SGP_CUDA_TRY(cudaStreamSynchronize(st));
            if (!(h.psf_sum > 0.0) || !std::isfinite(h.psf_sum)) return SGP_ERR_PSF;       // PAPER.md:27 needs a positive volume
            RowParams<T> P = row_params();
            P.submode = RFS_PSF; P.in0 = (const T *)psf[j]; P.cy = cy; P.cxs = cxs;
            P.spec = (C *)scratch;          // raw spectrum of this PSF
            if ((rc = launch_row(k_rowf[RF_SETUP], P, 1, st))) return rc;
            ColParams<T> Q = col_params();
            Q.in = (const C *)scratch; Q.out = (C *)scratch;
            if ((rc = launch_col(k_colf, Q, st))) return rc;
            khat_fixup_kernel<T><<<ew_grid(nspec), 256, 0, st>>>((const C *)scratch, khat + (size_t)j * nspec, khatB + (size_t)j * ny, ny, nx, G.C);
            launches++;
            SGP_CUDA_TRY(cudaGetLastError());
        }
        if (G.masked) {
            // alpha_j = A_j^T 1_S = IFFT2(conj K^_j FFT2(M_S)) (Eq.19 in reading A5), alpha = sum_j alpha_j, R by Eq.20
            for (int j = 0; j < p; ++j) {
                RowParams<T> P = row_params();
                P.submode = RFS_MASK_S;
                if ((rc = launch_row(k_rowf[RF_SETUP], P, 1, st))) return rc;
                ColParams<T> Q = col_params();
                Q.khat = khat + (size_t)j * nspec; Q.khatB = khatB + (size_t)j * ny; Q.p = 1;
                col_kernel_t<T> k1 = get_col<T>(Lc, CM_CONJSUM, false);
                SGP_CUDA_TRY(cudaFuncSetAttribute((const void *)k1, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)col_smem));
                if ((rc = launch_col(k1, Q, st))) return rc;
                RowParams<T> R = row_params();
                R.out0 = scratch; R.maskmode = MM_NONE;
                if ((rc = launch_row(k_rowi[RI_PLAIN], R, 1, st))) return rc;
                alpha_accum_kernel<T><<<ew_grid(n), 256, 0, st>>>(scratch, alpha, MR, n, opt.sigma_R, j == 0);
                launches++;
                SGP_CUDA_TRY(cudaMemcpyAsync(alphaJ + (size_t)j * n, scratch, n * sizeof(T), cudaMemcpyDeviceToDevice, st));
            }
            alpha_finish_kernel<T><<<ew_grid(n), 256, 0, st>>>(alpha, MR, alphaR, n);
            launches++;
            for (int j = 0; j < p; ++j) {     // alpha_j restricted to R (R needs all the alpha_j, Eq.20), in place
                alpha_finish_kernel<T><<<ew_grid(n), 256, 0, st>>>(alphaJ + (size_t)j * n, MR, alphaJ + (size_t)j * n, n);
                launches++;
            }
            SGP_CUDA_TRY(cudaGetLastError());
            std::vector<unsigned char> hm(n);
            SGP_CUDA_TRY(cudaMemcpyAsync(hm.data(), MR, n, cudaMemcpyDeviceToHost, st));
            SGP_CUDA_TRY(cudaStreamSynchronize(st));
            nR = 0;
            for (size_t i = 0; i < n; ++i) nR += hm[i];
        } else {
            nR = (long)n;
        }
        SGP_CUDA_TRY(cudaStreamSynchronize(st));
        psf_set = true;
        return SGP_OK;
    }

    int get_mask(unsigned char *maskR_out, void *alpha_out, long *nR_out, cudaStream_t st) override
    {
        if (!psf_set) return SGP_ERR_ARG;
        if (G.masked) {
            if (maskR_out) SGP_CUDA_TRY(cudaMemcpyAsync(maskR_out, MR, n, cudaMemcpyDeviceToDevice, st));
            if (alpha_out) SGP_CUDA_TRY(cudaMemcpyAsync(alpha_out, alpha, n * sizeof(T), cudaMemcpyDeviceToDevice, st));
        } else {
            if (maskR_out) SGP_CUDA_TRY(cudaMemsetAsync(maskR_out, 1, n, st));
            if (alpha_out) {
                std::vector<T> h(n, (T)p);
                SGP_CUDA_TRY(cudaMemcpyAsync(alpha_out, h.data(), n * sizeof(T), cudaMemcpyHostToDevice, st));
            }
        }
        SGP_CUDA_TRY(cudaStreamSynchronize(st));
        if (nR_out) *nR_out = nR;
        return SGP_OK;
    }

    // out = A_j x (Eq.16) or A_j^T x (Eq.17)
    int apply(bool transpose, int j, const void *x, void *out, cudaStream_t st) override
    {
        if (!psf_set || j < 0 || j >= p || !x || !out) return SGP_ERR_ARG;
        int rc;
        RowParams<T> P = row_params();
        P.in0 = (const T *)x; P.maskmode = transpose ? MM_S : MM_R;
        if ((rc = launch_row(k_rowf[RF_PLAIN], P, 1, st))) return rc;
        ColParams<T> Q = col_params();
        Q.khat = khat + (size_t)j * nspec; Q.khatB = khatB + (size_t)j * ny; Q.p = 1;
        col_kernel_t<T> k1 = get_col<T>(Lc, transpose ? CM_CONJSUM : CM_MULT, false);
        SGP_CUDA_TRY(cudaFuncSetAttribute((const void *)k1, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)col_smem));
        if ((rc = launch_col(k1, Q, st))) return rc;
        RowParams<T> R = row_params();
        R.out0 = scratch; R.maskmode = transpose ? MM_R : MM_S;
        if ((rc = launch_row(k_rowi[RI_PLAIN], R, 1, st))) return rc;
        SGP_CUDA_TRY(cudaMemcpyAsync(out, scratch, n * sizeof(T), cudaMemcpyDeviceToDevice, st));
        SGP_CUDA_TRY(cudaStreamSynchronize(st));
        return SGP_OK;
    }

    int rfft2(const void *x, void *spec_out, cudaStream_t st) override
    {
        if (!x || !spec_out) return SGP_ERR_ARG;
        int rc;
        RowParams<T> P = row_params();
        P.in0 = (const T *)x;
        if ((rc = launch_row(k_rowf[RF_PLAIN], P, 1, st))) return rc;
        ColParams<T> Q = col_params();
        if ((rc = launch_col(k_colf, Q, st))) return rc;
        spec_to_rfft2_kernel<T><<<ew_grid(n), 256, 0, st>>>(spec, (C *)spec_out, ny, nx, G.C);
        launches++;
        SGP_CUDA_TRY(cudaGetLastError());
        SGP_CUDA_TRY(cudaStreamSynchronize(st));
        return SGP_OK;
    }
    int irfft2(const void *spec_in, void *x_out, cudaStream_t st) override
    {
        if (!spec_in || !x_out) return SGP_ERR_ARG;
        int rc;
        rfft2_to_spec_kernel<T><<<ew_grid(nspec), 256, 0, st>>>((const C *)spec_in, spec, ny, nx, G.C, (T)(1.0 / ((double)ny * (double)nx)));
        launches++;
        SGP_CUDA_TRY(cudaGetLastError());
        col_kernel_t<T> ki = get_col<T>(Lc, CM_INV, false);
        SGP_CUDA_TRY(cudaFuncSetAttribute((const void *)ki, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)col_smem));
        ColParams<T> Q = col_params();
        if ((rc = launch_col(ki, Q, st))) return rc;
        RowParams<T> R = row_params();
        R.out0 = (T *)x_out; R.maskmode = MM_NONE;
        if ((rc = launch_row(k_rowi[RI_PLAIN], R, 1, st))) return rc;
        SGP_CUDA_TRY(cudaStreamSynchronize(st));
        return SGP_OK;
    }

    int run(int algorithm, const void *const *g, const void *const *b_arr, const double *b_const,
            const void *f0, void *f_out, const sgp_options *ropt, sgp_result *res, cudaStream_t st) override;
    int run_batched(int algorithm, const void *const *g, const void *const *b_arr, const double *b_const,
                    const void *const *f0, void *const *f_out, const sgp_options *ropt, sgp_result *res, cudaStream_t st) override;
    int ensure_trace(int max_iter, const sgp_result *res, Trace *tr, cudaStream_t st);
    int enqueue_sgp_iteration(const RowParams<T> &Pbase, const DevOpts &o, const Trace &tr, const double *bconst, int b_is_array, cudaStream_t st);
    int enqueue_ratio(const RowParams<T> &Pbase, int lazy, cudaStream_t st);
    int enqueue_rl_round(const DevOpts &o, const Trace &tr, const double *bconst, int b_is_array, cudaStream_t st);
    int enqueue_osem_cycle(const DevOpts &o, const Trace &tr, const double *bconst, int b_is_array, cudaStream_t st);
    int enqueue_many(int algorithm, int count, const RowParams<T> &Pb, const DevOpts &o, const Trace &tr, const double *bconst,
                     int b_is_array, cudaStream_t st);
};

}  // namespace sgpk
