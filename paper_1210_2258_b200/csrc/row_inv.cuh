// row_inv.cuh -- half spectrum -> real rows (row pass of the inverse FFT2).  The epilogue modes (row_epi.cuh) carry
// steps a3 + a5 + a6 (gradient, BB sums, step length) with the lazy f update of a10, a9 (line-search sum at
// lambda = 1, Armijo test, book-keeping), the start-point / RL objective, the adaptive bounds and the RL update.
// Same thread organisation as row_fwd.cuh: the TF threads of a row synchronise only among themselves.
#pragma once
#include "row_epi.cuh"
#include "row_fwd.cuh"

namespace sgpk {

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
__global__ void __launch_bounds__(256, 2) row_inv_kernel(const RowParams<T> P)
{
    using C = cx<T>;
    constexpr int E = fft_E<T>(L);
    constexpr int TF = L / E;
    constexpr int RS = fft_padded_len(L, E);
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ double red[kNQ * 32];
    C *sm = reinterpret_cast<C *>(smem_raw);
    pdl_trigger();
    pdl_wait();
    // the stop flag is tested only after the loads of the spectrum have been issued (all stores come later)
    const int stop = P.check_status ? P.ct->status : 0;

    const Geom &G = P.G;
    const int tid = threadIdx.x;
    const int row = tid / TF, t = tid - row * TF;
    const int y = blockIdx.x * G.RB + row;
    const int j = blockIdx.y;
    constexpr int nx = 2 * L;
    C *smrow = sm + row * RS;
    const SyncGroup<TF> sync{1 + row};
    // ---- tile-major spectrum -> re-tangled Z in shared memory, one (k, L-k) pair per step, k = t + TF i;
    //      Z[0] = (X0 + XL) + i (X0 - XL);  Z[L/2] = 2 conj X[L/2]
    {
        const C *src = P.spec + (size_t)j * P.specplane;
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
#pragma unroll
            for (int i = 1; i < E / 2; ++i) {
                const int k = t + TF * i;
                C zk, zlk;
                retangle<T>(pa[(size_t)i * stride], *(pb - (size_t)i * stride), __ldg(&P.twh[k]), zk, zlk);
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
    sync();
    {
        C v[E];
#pragma unroll
        for (int e = 0; e < E; ++e) v[e] = smrow[fft_pad<E>(t + TF * e)];
        fft_block<T, L, E, +1>(v, smrow, 1, t, P.tw, sync);
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
        if (P.submode == RIP_STORE) {
            epi_store<T, L, TF, MK>(P, wrow, t, y, rowbase, base);
        } else {
            // RIP_RLMINMAX: adaptive bounds from one RL step (A19)
            double acc[2] = {-INFINITY, -INFINITY};   // (-min positive, max)
            epi_rl<T, L, TF, false, MK>(P, wrow, t, rowbase, acc);
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
            if (publish_partials<2>(acc, P.part, bid, nblk, &P.ct->counter[TK_MINMAX])) {
                if (tid == 0) {
                    double mn = -INFINITY, mx = -INFINITY;
                    for (unsigned int b = 0; b < nblk; ++b) { mn = fmax(mn, __ldcg(&P.part[2 * b])); mx = fmax(mx, __ldcg(&P.part[2 * b + 1])); }
                    const double ymin = -mn, ymax = mx;
                    if (!(ymin < INFINITY) || !(ymax > 0.0)) P.ct->status = SGP_ERR_DATA;
                    else if (ymax / ymin < 50.0) { P.ct->L1 = ymin / 10.0; P.ct->L2 = ymax * 10.0; }
                    else                         { P.ct->L1 = ymin;        P.ct->L2 = ymax; }
                }
            }
        }
    } else if constexpr (MODE == RI_GRAD) {
        double acc[4] = {0.0, 0.0, 0.0, 0.0};
        epi_grad<T, L, TF, MK>(P, wrow, t, rowbase, acc);
        block_reduce_sum<4>(acc, red);
        if (publish_partials<4>(acc, P.part, bid, nblk, &P.ct->counter[TK_GRAD])) {
            final_sum<4>(acc, P.part, nblk, red);
            if (tid == 0) { P.ct->pending = 0; bb_step(P.ct, P.o, P.tr, acc[0], acc[1], acc[2], acc[3]); }   // a6
        }
    } else if constexpr (MODE == RI_LS || MODE == RI_QJ || MODE == RI_LSF) {
        constexpr bool LS = (MODE == RI_LS || MODE == RI_LSF), SPEC = (MODE == RI_LSF);
        const bool plain = (MODE == RI_QJ) && P.submode == QJ_PLAIN;
        double acc[1] = {0.0};
        // SGP loop: q is double-buffered; this kernel reads buffer qsel and (SPEC) writes q + u into the other one
        const int sel = LS ? P.ct->qsel : 0;
        const T *qin = P.in1 + (size_t)sel * P.qbuf;
        T *qout = SPEC ? const_cast<T *>(P.in1) + (size_t)(sel ^ 1) * P.qbuf : nullptr;
        T *wmut = reinterpret_cast<T *>(smrow);
        epi_kl<T, L, TF, LS, MK, SPEC>(P, wrow, wmut, qin, qout, t, y, j, base, plain, acc);
        if (plain) return;
        block_reduce_sum<1>(acc, red);
        const int tk = LS ? TK_LS : TK_QJ;
        if (publish_partials<1>(acc, P.part, bid, nblk, &P.ct->counter[tk])) {
            final_sum<1>(acc, P.part, nblk, red);
            const double J = acc[0];
            Ctrl *ct = P.ct;
            if constexpr (LS) {
                double gd[1];
                final_sum<1>(gd, P.part2, gridDim.x, red);     // grad'd partials of the projection kernel
                if (tid == 0) {
                    // Alg.1 step 5 at lambda = 1: J(f + d) <= J_ref + beta * 1 * grad'd
                    const double Jref = armijo_ref(ct);
                    ct->gd = gd[0]; ct->Jref = Jref; ct->Jtrial = J;
                    int acc1 = (isfinite(J) && J <= Jref + P.o.beta * gd[0]) ? 1 : 0;
                    if (P.tr.force_lambda) {
                        const double fl = P.tr.force_lambda[ct->k];
                        if (isfinite(fl)) acc1 = (fl == 1.0) ? 1 : 0;
                    }
                    ct->accepted = acc1;
                    // a10 (book-keeping; f is updated lazily by K3), a11.  SPEC: q(k+1) and the ratio spectrum are
                    // already in place, so the ratio kernel of the next iteration has nothing to do.
                    if (acc1) finish_iteration(ct, P.o, P.tr, 1.0, J, 0, SPEC ? 0 : 2);
                }
            } else if (tid == 0) {
                if (P.submode == QJ_INIT) {
                    ct->J = J; ct->Jhist[0] = J; ct->nJ = 1;
                    if (P.tr.J) P.tr.J[0] = J;
                    if (!isfinite(J)) ct->status = SGP_ERR_NONFINITE;
                } else {   // QJ_RL: J0(f(k)) and the stopping rules before the k-th RL update
                    const int k = ct->k;
                    const double Jold = ct->J;
                    ct->J = J;
                    if (P.tr.J) P.tr.J[k] = J;
                    if (!isfinite(J)) ct->status = SGP_ERR_NONFINITE;
                    else {
                        int r = stop_test(P.o, k, J, Jold, k > 0);
                        if (r) ct->status = r; else ct->k = k + 1;
                    }
                }
            }
        }
        if constexpr (SPEC) {
            // a1 of the next iteration, speculating on lambda = 1: forward row transform of the ratio parked in shared
            // memory by the epilogue; the spectrum row this warp read at the top is overwritten in place
            C v[E];
            sync();
#pragma unroll
            for (int e = 0; e < E; ++e) v[e] = smrow[t + TF * e];
            fwd_fft_store<T, L>(v, smrow, t, sync, P, y, j);
        }
    } else {   // RI_RLUPDATE, a12: f <- (M_R/alpha) o f o sum_j A_j^T(g_j/(A_j f + b_j))   (Eq.1/13/21)
        double dummy[2];
        epi_rl<T, L, TF, true, MK>(P, wrow, t, rowbase, dummy);
    }
}

}  // namespace sgpk
