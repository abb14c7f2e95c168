// row_inv.cuh -- half spectrum -> real rows (row pass of the inverse FFT2).  The epilogue modes (row_epi.cuh) carry
// steps a3 + a5 + a6 (gradient, BB sums, step length) with the lazy f update of a10, a9 (line-search sum at
// lambda = 1, Armijo test, book-keeping), the start-point / RL objective, the adaptive bounds and the RL update.
// Same thread organisation as row_fwd.cuh: the TF threads of a row synchronise only among themselves.
#pragma once
#include "row_epi.cuh"
#include "row_fwd.cuh"

namespace sgpk {

// L2 prefetch of the plane rows the epilogue streams, issued once the spectrum row has landed, i.e. while the transform computes
// (single-wave kernels: without it DRAM idles during the transforms and every warp asks for its rows at the same moment).
// 0 = off; 2 = the line-search kernels only (g_j, q_j): K6 35.3 -> 33.1 us at 2048^2, 95.0 -> 93.0 us at 3 x 2048^2; 1 = also the
// gradient kernel (f, d, grad(k-1): 28.5 -> 28.7 us), the RL ratio kernel (27.9 -> 28.7 us) and the RL update: slower, so 2 it is;
// 3 = 2 + the RL update kernel (no change).  Requested at the top of the kernel the rows compete with the spectrum loads (round 1:
// K3 + 10 %).
#ifndef SGP_EPI_PF
#define SGP_EPI_PF 2
#endif
// the nx elements of one plane row, 128-byte lines spread over the TF lanes of the row
template <typename T, int TF> __device__ __forceinline__ void prefetch_row(const T *row, int nx, int t)
{
    const char *b = reinterpret_cast<const char *>(row);
    const int bytes = nx * (int)sizeof(T);
    for (int o = t * 128; o < bytes; o += TF * 128) prefetch_l2(b + o);
}

// re-tangling of one (k, L-k) pair: a = X[k], b = conj X[L-k], w = exp(-2 pi i k/nx):
//   S = a + b, Tm = i conj(w) (a - b):  Z[k] = S + Tm, Z[L-k] = conj(S - Tm)
template <typename T> __device__ __forceinline__ void retangle(cx<T> a, cx<T> xb, cx<T> w, cx<T> &zk, cx<T> &zlk)
{
    const cx<T> b = cconj(xb);
    const cx<T> Sk = cadd(a, b), Dk = csub(a, b);
    const cx<T> Tm = cmulc(mk<T>(-Dk.y, Dk.x), w);
    zk = cadd(Sk, Tm);
    zlk = cconj(csub(Sk, Tm));
}

template <typename T, int L, int MODE, bool MK>
__global__ void __launch_bounds__(256, SGP_ROW_MINB) row_inv_kernel(const RowParams<T> P)
{
    using C = cx<T>;
    constexpr int E = fft_E<T>(L);
    constexpr int TF = L / E;
    constexpr int RS = row_stride(L, E);
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ double red[kNQ * 32];
    C *sm = reinterpret_cast<C *>(smem_raw);
    pdl_trigger();
    pdl_wait();
    RowPtrs<T> X = row_ptrs(P);                                  // this problem's arrays (batched plans: blockIdx.z)
    // the stop flag is tested only after the loads of the spectrum have been issued (all stores come later)
    const int stop = P.check_status ? X.ct->status : 0;
    if constexpr (MODE == RI_QJ) { if (P.submode == QJ_REFRESH && X.ct->refresh_due == 0) return; }      // A21: only after every n-th iteration

    const Geom &G = P.G;
    const int tid = threadIdx.x;
    constexpr int TFP = group_threads(TF);                       // threads per row incl. padding lanes (5-smooth lengths)
    const int row = tid / TFP, traw = tid - row * TFP;
    const bool act = TFP == TF ? true : traw < TF;
    const int t = TFP == TF ? traw : (traw < TF ? traw : TF - 1);
    X.act = act;
    const int y = blockIdx.x * G.RB + row;
    const int j = blockIdx.y;
    constexpr int nx = 2 * L;
    C *smrow = sm + row * RS;
    const SyncGroup<TFP> sync{1 + row};
    // twiddle tables in shared memory (row_fwd.cuh): wanted from the inverse transform on; the re-tangling below, which
    // starts at once, reads exp(-2 pi i k/nx) from global memory
    constexpr bool TWS = SGP_TW_SMEM != 0;
    C *tw_s = sm + (size_t)G.RB * RS;
    const C *tw = TWS ? tw_s : P.tw, *twh = TWS ? tw_s + even_up(tw_total(L, E)) : P.twh;
    if constexpr (TWS) { if (stop == 0) row_tables_issue<T, L>(tw_s, P, tid, (int)blockDim.x); }
    // ---- tile-major spectrum -> re-tangled Z in shared memory, one (k, L-k) pair per step, k = t + TF i;
    //      Z[0] = (X0 + XL) + i (X0 - XL);  Z[L/2] = 2 conj X[L/2]
    {
        const C *src = X.spec + (size_t)j * P.specplane;
        {   // i = 0
            const C a = src[spec_index(G, y, t)];
            if (t == 0) {
                smrow[0] = mk<T>(a.x + a.y, a.x - a.y);
                const C m = src[spec_index(G, y, L / 2)];
                smrow[fft_pad<E>(L / 2)] = mk<T>((T)2 * m.x, (T)-2 * m.y);
            } else {
                C zk, zlk;
                retangle<T>(a, src[spec_index(G, y, L - t)], __ldg(&P.twh[t]), zk, zlk);
                smrow[fft_pad<E>(t)] = zk;
                smrow[fft_pad<E>(L - t)] = zlk;
            }
        }
        if ((TF & (G.C - 1)) == 0) {
            // TF is a multiple of the tile width: kx -> kx + TF moves TF/C tiles on, i.e. TF*ny elements
            const size_t stride = (size_t)TF * (size_t)G.ny;
            const C *pa = src + spec_index(G, y, t);
            const C *pb = src + spec_index(G, y, L - TF - t) + stride;
            C wt = mk<T>((T)1, (T)0);
            if constexpr (kRowTwc<T, E>) wt = __ldg(&P.twh[t]);
#pragma unroll
            for (int i = 1; i < E / 2; ++i) {
                const int k = t + TF * i;
                C zk, zlk;
                C wk;
                if constexpr (kRowTwc<T, E>) wk = cmul(wt, twc_const<T, E>(i)); else wk = __ldg(&P.twh[k]);
                retangle<T>(pa[(size_t)i * stride], *(pb - (size_t)i * stride), wk, zk, zlk);
                smrow[fft_pad<E>(k)] = zk;
                smrow[fft_pad<E>(L - k)] = zlk;
            }
        } else {
#pragma unroll 4
            for (int i = 1; i < E / 2; ++i) {
                const int k = t + TF * i;
                C zk, zlk;
                retangle<T>(src[spec_index(G, y, k)], src[spec_index(G, y, L - k)], __ldg(&P.twh[k]), zk, zlk);
                smrow[fft_pad<E>(k)] = zk;
                smrow[fft_pad<E>(L - k)] = zlk;
            }
        }
    }
    if (stop != 0) return;
    if constexpr (TWS) row_tables_wait(); else sync();
    if constexpr (SGP_EPI_PF != 0 && sizeof(T) == 4) {
        // the spectrum row has landed: start the plane rows of the epilogue on their way to L2 while the transform computes
        // (requested at the top of the kernel they compete with the spectrum loads, which the transform waits for)
        const size_t rb = (size_t)y * nx, bs = (size_t)j * P.plane + rb;
        if constexpr (MODE == RI_GRAD && SGP_EPI_PF == 1) {
            prefetch_row<T, TF>(X.in0 + rb, nx, t); prefetch_row<T, TF>(X.in1 + rb, nx, t); prefetch_row<T, TF>(X.out0 + rb, nx, t);
        } else if constexpr (MODE == RI_LS || MODE == RI_LSF) {
            prefetch_row<T, TF>(X.in0 + bs, nx, t);
            prefetch_row<T, TF>(X.in1 + (size_t)X.ct->qsel * P.qbuf + bs, nx, t);
        } else if constexpr ((MODE == RI_QJ || MODE == RI_QJF) && SGP_EPI_PF == 1) {
            prefetch_row<T, TF>(X.in0 + bs, nx, t);
        } else if constexpr ((MODE == RI_RLUPDATE || MODE == RI_RLUPF) && (SGP_EPI_PF == 1 || SGP_EPI_PF == 3)) {
            prefetch_row<T, TF>(X.in0 + rb, nx, t);
        }
    }
    {
        C v[E];
#pragma unroll
        for (int e = 0; e < E; ++e) v[e] = smrow[fft_pad<E>(t + TF * e)];
        fft_block<T, L, E, +1, TWS, kRowTwp<T>>(v, smrow, 1, t, tw, sync);
        // park the row (w(y, 2m), w(y, 2m+1)), m = t + TF e, in natural order (no padding) for the epilogue
        sync();
#pragma unroll
        for (int e = 0; e < E; ++e) smrow[t + TF * e] = v[e];
        sync();
    }

    const T *wrow = reinterpret_cast<const T *>(smrow);
    const size_t rowbase = (size_t)y * nx;
    const size_t base = (size_t)j * P.plane + rowbase;
    const unsigned int nblk = gridDim.x * gridDim.y;
    const int bid = blockIdx.y * gridDim.x + blockIdx.x;

    if constexpr (MODE == RI_PLAIN) {
        if (P.submode == RIP_STORE || P.submode == RIP_STORE_POS) {
            epi_store<T, L, TF, MK>(P, X, wrow, t, y, rowbase, base);
        } else {
            // RIP_RLMINMAX: adaptive bounds from one RL step (A19)
            double acc[2] = {-INFINITY, -INFINITY};   // (-min positive, max)
            epi_rl<T, L, TF, false, MK>(P, X, wrow, t, rowbase, acc);
            // max-reduction over the block (fixed tree)
            const int lane = tid & 31, wid = tid >> 5, nw = (blockDim.x + 31) >> 5;
#pragma unroll
            for (int q = 0; q < 2; ++q) {
#pragma unroll
                for (int off = 16; off > 0; off >>= 1) acc[q] = fmax(acc[q], __shfl_down_sync(0xffffffffu, acc[q], off));
                if (lane == 0) red[q * 32 + wid] = acc[q];
            }
            __syncthreads();
            if (tid == 0) {
                for (int q = 0; q < 2; ++q) { double m = red[q * 32]; for (int w = 1; w < nw; ++w) m = fmax(m, red[q * 32 + w]); acc[q] = m; }
            }
            __syncthreads();
            if (publish_partials<2>(acc, X.part, bid, nblk, &X.ct->counter[TK_MINMAX])) {
                if (tid == 0) {
                    double mn = -INFINITY, mx = -INFINITY;
                    for (unsigned int b = 0; b < nblk; ++b) { mn = fmax(mn, __ldcg(&X.part[2 * b])); mx = fmax(mx, __ldcg(&X.part[2 * b + 1])); }
                    const double ymin = -mn, ymax = mx;
                    if (!(ymin < INFINITY) || !(ymax > 0.0)) X.ct->status = SGP_ERR_DATA;
                    else if (ymax / ymin < 50.0) { X.ct->L1 = ymin / 10.0; X.ct->L2 = ymax * 10.0; }
                    else                         { X.ct->L1 = ymin;        X.ct->L2 = ymax; }
                }
            }
        }
    } else if constexpr (MODE == RI_GRAD) {
        double acc[4] = {0.0, 0.0, 0.0, 0.0};
        epi_grad<T, L, TF, MK>(P, X, wrow, t, rowbase, acc);
        if (!act) { acc[0] = 0.0; acc[1] = 0.0; acc[2] = 0.0; acc[3] = 0.0; }     // padding lanes repeat lane TF - 1
        block_reduce_sum<4>(acc, red);
        if (publish_partials<4>(acc, X.part, bid, nblk, &X.ct->counter[TK_GRAD])) {
            final_sum<4>(acc, X.part, nblk, red);
            if (tid == 0) { X.ct->pending = 0; bb_step(X.ct, P.o, X.tr, acc[0], acc[1], acc[2], acc[3]); }   // a6
        }
    } else if constexpr (MODE == RI_LS || MODE == RI_QJ || MODE == RI_LSF || MODE == RI_QJF) {
        constexpr bool LS = (MODE == RI_LS || MODE == RI_LSF), SPEC = (MODE == RI_LSF);
        constexpr bool RATIO = (MODE == RI_LSF || MODE == RI_QJF);
        const bool plain = (MODE == RI_QJ || MODE == RI_QJF) && P.submode == QJ_PLAIN;
        double acc[1] = {0.0};
        // SGP loop: q is double-buffered; this kernel reads buffer qsel and (SPEC) writes q + u into the other one
        const int sel = LS ? X.ct->qsel : 0;
        const T *qin = X.in1 + (size_t)sel * P.qbuf;
        T *qout = SPEC ? const_cast<T *>(X.in1) + (size_t)(sel ^ 1) * P.qbuf : nullptr;
        T *wmut = reinterpret_cast<T *>(smrow);
        // where the row itself goes: u_j (SGP), q_j (set-up, RL); the refresh round (A21) rewrites the current q buffer
        T *rowout = X.out0;
        if (MODE == RI_QJ && P.submode == QJ_REFRESH) rowout += (size_t)X.ct->qsel * P.qbuf;
        epi_kl<T, L, TF, LS, MK, RATIO, MODE != RI_QJF, SPEC>(P, X, wrow, wmut, qin, qout, rowout, t, y, j, base, plain, acc);
        if (!act) acc[0] = 0.0;                                    // padding lanes repeat lane TF - 1
        if (!plain) {
        block_reduce_sum<1>(acc, red);
        const int tk = LS ? TK_LS : TK_QJ;
        if (publish_partials<1>(acc, X.part, bid, nblk, &X.ct->counter[tk])) {
            final_sum<1>(acc, X.part, nblk, red);
            const double J = acc[0];
            Ctrl *ct = X.ct;
            if constexpr (LS) {
                double gd[1];
                final_sum<1>(gd, X.part2, gridDim.x, red);     // grad'd partials of the projection kernel
                if (tid == 0) {
                    // Alg.1 step 5 at lambda = 1: J(f + d) <= J_ref + beta * 1 * grad'd
                    const double Jref = armijo_ref(ct);
                    ct->gd = gd[0]; ct->Jref = Jref; ct->Jtrial = J;
                    int acc1 = (isfinite(J) && J <= Jref + P.o.beta * gd[0]) ? 1 : 0;
                    if (X.tr.force_lambda) {
                        const double fl = X.tr.force_lambda[ct->k];
                        if (isfinite(fl)) acc1 = (fl == 1.0) ? 1 : 0;
                    }
                    ct->accepted = acc1;
                    // re-arm the backtracking prologue of the ratio kernel that follows (aux.cuh: backtrack_rounds)
                    if (X.btsync) { X.btsync[kBtNext] = 0; X.btsync[kBtDone] = 0; X.btsync[kBtDecided] = 0; X.btsync[kBtFinal] = 0; }
                    if (!acc1 && P.o.max_backtracks < 1 && !X.tr.force_lambda) { ct->status = SGP_ERR_LINESEARCH; ct->accepted = 1; }   // A16
                    // a10 (book-keeping; f is updated lazily by K3), a11.  SPEC: q(k+1) and the ratio spectrum are
                    // already in place, so the ratio kernel of the next iteration has nothing to do.
                    if (acc1) finish_iteration(ct, P.o, X.tr, 1.0, J, 0, SPEC ? 0 : 2);
                }
            } else if (tid == 0) {
                if (P.submode == QJ_INIT) {
                    ct->J = J; ct->Jhist[0] = J; ct->nJ = 1;
                    if (X.tr.J) X.tr.J[0] = J;
                    if (!isfinite(J)) ct->status = SGP_ERR_NONFINITE;
                } else if (P.submode == QJ_REFRESH) {
                    // A21: J0(f(k)) recomputed from f replaces the value carried by q + lambda u; the stopping rules that
                    // finish_iteration left to this kernel
                    const int k = ct->k;
                    ct->J = J; ct->Jhist[k % P.o.armijo_memory] = J;
                    if (X.tr.J) X.tr.J[k] = J;
                    ct->refresh_due = 0;
                    if (!isfinite(J)) ct->status = SGP_ERR_NONFINITE;
                    else { int r = stop_test(P.o, k, J, ct->Jprev, true); if (r) ct->status = r; }
                } else {   // QJ_RL: J0(f(k)) and the stopping rules before the k-th RL update
                    const int k = ct->k;
                    const double Jold = ct->J;
                    ct->J = J;
                    if (X.tr.J) X.tr.J[k] = J;
                    if (!isfinite(J)) ct->status = SGP_ERR_NONFINITE;
                    else {
                        int r = stop_test(P.o, k, J, Jold, k > 0);
                        if (r) ct->status = r; else ct->k = k + 1;
                    }
                }
            }
        }
        }   // !plain
        if constexpr (RATIO) {
            // a1 of the next step (SGP: speculating on lambda = 1): forward row transform of the ratio parked in shared
            // memory by the epilogue; the spectrum row this warp read at the top is overwritten in place
            C v[E];
            sync();
#pragma unroll
            for (int e = 0; e < E; ++e) v[e] = smrow[t + TF * e];
            fwd_fft_store<T, L, TWS>(v, smrow, t, sync, P, X, y, j, tw, twh);
        }
    } else if constexpr (MODE == RI_RLUPDATE) {   // a12: f <- (M_R/alpha) o f o sum_j A_j^T(g_j/(A_j f + b_j))   (Eq.1/13/21)
        double dummy[2];
        epi_rl<T, L, TF, true, MK>(P, X, wrow, t, rowbase, dummy);
    } else {   // RI_RLUPF: a12 and the forward row transform of the new f (the first pass of A_j f of the next round)
        double dummy[2];
        epi_rl<T, L, TF, true, MK, true>(P, X, wrow, t, rowbase, dummy, reinterpret_cast<T *>(smrow));
        C v[E];
        sync();
#pragma unroll
        for (int e = 0; e < E; ++e) v[e] = smrow[t + TF * e];
        fwd_fft_store<T, L, TWS>(v, smrow, t, sync, P, X, y, 0, tw, twh);
    }
    // n_fft2 (include/sgp.h): the two-dimensional transforms this launch and the column pass before it completed
    if (P.count_fft && bid == 0 && tid == 0) atomicAdd(&X.ct->nfft, (unsigned long long)P.count_fft);
}

}  // namespace sgpk
