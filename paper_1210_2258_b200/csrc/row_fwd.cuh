// row_fwd.cuh -- real rows -> half spectrum (row pass of FFT2), with the elementwise work of the iteration
// fused into the load stage.
//
// One row is transformed by TF = L/E threads (a warp for the 2048-wide grid: L = 1024, E = 32, passes 32 x 32);
// the threads of a row synchronise only among themselves (SyncGroup), so the rows of a CTA drift apart and
// the loads of one row overlap the butterflies and stores of another.  grid = (ny/RB, images), block = RB*TF
// threads, dynamic smem = RB * padded(L) complex.
#pragma once
#include "ew.cuh"
#include "aux.cuh"

namespace sgpk {

// pairs loaded ahead of the first store of a batch in the load stage
template <typename T> __host__ __device__ constexpr int fwd_batch(int E)
{
    return sizeof(T) == 8 ? (E % 4 == 0 ? 4 : 2) : (E % 8 == 0 ? 8 : 4);
}

// Shared-memory copies of the twiddle tables of a row kernel (fft_core.cuh: SGP_TW_SMEM), behind the rows' lines:
// the pass tables of the length-L complex FFT and exp(-2 pi i k/nx), k <= L/2, of the real<->complex step.  The copy is
// asynchronous (cp.async, 16 bytes per request, no registers): issued at the start of the kernel, awaited before the
// first use.  Counts are rounded up to even numbers (the device tables are allocated with that padding).
__host__ __device__ constexpr int even_up(int n) { return (n + 1) & ~1; }
template <typename T> __host__ __device__ constexpr size_t row_table_entries(int L)
{
    return SGP_TW_SMEM ? (size_t)even_up(tw_total(L, fft_E<T>(L))) + (size_t)even_up(L / 2 + 1) : 0;
}
template <typename T, int L>
__device__ __forceinline__ void row_tables_issue(cx<T> *tw_s, const RowParams<T> &P, int tid, int nthr)
{
    constexpr int E = fft_E<T>(L);
    constexpr int N1 = even_up(tw_total(L, E)), N2 = even_up(L / 2 + 1);
    constexpr int per16 = 16 / (int)sizeof(cx<T>);               // complex numbers per 16-byte request: 2 (float) or 1 (double)
    const unsigned int s1 = (unsigned int)__cvta_generic_to_shared(tw_s), s2 = (unsigned int)__cvta_generic_to_shared(tw_s + N1);
    for (int i = tid; i < N1 / per16; i += nthr)
        asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(s1 + 16u * i), "l"(reinterpret_cast<const char *>(P.tw) + 16 * (size_t)i) : "memory");
    for (int i = tid; i < N2 / per16; i += nthr)
        asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(s2 + 16u * i), "l"(reinterpret_cast<const char *>(P.twh) + 16 * (size_t)i) : "memory");
    asm volatile("cp.async.commit_group;" ::: "memory");
}
// all threads of the CTA: the tables have landed and are visible
__device__ __forceinline__ void row_tables_wait()
{
    asm volatile("cp.async.wait_all;" ::: "memory");
    __syncthreads();
}

// untangling of one (k, L-k) pair: a = Z[k], zb = Z[L-k], w = exp(-2 pi i k/nx):
//   E = (a + conj zb)/2, O = -i (a - conj zb)/2:  X[k] = E + w O,  X[L-k] = conj(E - w O)
template <typename T> __device__ __forceinline__ void untangle(cx<T> a, cx<T> zb, cx<T> w, cx<T> &xk, cx<T> &xlk)
{
    const cx<T> b = cconj(zb);
    const cx<T> Ek = mk<T>((T)0.5 * (a.x + b.x), (T)0.5 * (a.y + b.y));
    const cx<T> Dk = mk<T>((T)0.5 * (a.x - b.x), (T)0.5 * (a.y - b.y));
    const cx<T> wo = cmul(w, mk<T>(Dk.y, -Dk.x));          // w * (-i Dk)
    xk = cadd(Ek, wo);
    xlk = cconj(csub(Ek, wo));
}

// Forward transform of one row held as v[e] = (x[2m], x[2m+1]), m = t + TF e, by the TF threads of the row, and
// store of its half spectrum (tile-major).  Shared by the forward row kernel and the fused line-search kernel.
// tw / twh: the tables, in shared memory when TWS
#ifndef SGP_ROW_TWP
#define SGP_ROW_TWP 0      // option: pass twiddles of the float row transforms from a few table entries and one product each (fft_core.cuh: TWP); off, see col.cuh
#endif
#ifndef SGP_TWP_F64
#define SGP_TWP_F64 0
#endif
template <typename T> constexpr bool kRowTwp = SGP_ROW_TWP && (sizeof(T) == 4 || SGP_TWP_F64);
// experiment: exp(-2 pi i k/nx), k = t + TF i, of the real<->complex step as (table entry t) x (constant exp(-i pi i/E)): one load
// and E/2 - 1 products with immediates instead of E/2 loads (float, 32 or 16 elements per thread, tile width dividing TF)
#ifndef SGP_ROW_TWC
#define SGP_ROW_TWC 0
#endif
template <typename T, int E> constexpr bool kRowTwc = SGP_ROW_TWC && sizeof(T) == 4 && (E == 32 || E == 16);
// exp(-i pi i / E), i < E/2
template <typename T, int E> __device__ __forceinline__ cx<T> twc_const(int i)
{
    if constexpr (E == 32) return mk<T>((T)cos64q(i), (T)-sin64q(i));
    else return mk<T>((T)cos32(i), (T)-sin32(i));
}
template <typename T, int L, bool TWS, typename SYNC>
__device__ __forceinline__ void fwd_fft_store(cx<T> (&v)[fft_E<T>(L)], cx<T> *smrow, const int t, const SYNC &sync,
                                              const RowParams<T> &P, const RowPtrs<T> &X, const int y, const int j, const cx<T> *tw, const cx<T> *twh)
{
    using C = cx<T>;
    constexpr int E = fft_E<T>(L);
    constexpr int TF = L / E;
    const Geom &G = P.G;
    // ---- complex FFT of length L = nx/2 over z[m] = x[2m] + i x[2m+1]
    fft_block<T, L, E, -1, TWS, kRowTwp<T>>(v, smrow, 1, t, tw, sync);
    sync();
#pragma unroll
    for (int e = 0; e < E; ++e) smrow[fft_pad<E>(t + TF * e)] = v[e];
    sync();

    // ---- untangle the two interleaved real transforms, one (k, L-k) pair per step, and store tile-major:
    //      E = (Z[k] + conj Z[L-k])/2, O = -i (Z[k] - conj Z[L-k])/2, w = exp(-2 pi i k/nx):
    //      X[k] = E + w O,  X[L-k] = conj(E - w O);  entry 0 = (X[0], X[L]) packed;  X[L/2] = conj Z[L/2]
    C *dst = X.spec + (size_t)j * P.specplane;
    {   // i = 0
        const C a = smrow[fft_pad<E>(t)];
        if (t == 0) {
            if (X.act) { dst[spec_index(G, y, 0)] = mk<T>(a.x + a.y, a.x - a.y); dst[spec_index(G, y, L / 2)] = cconj(smrow[fft_pad<E>(L / 2)]); }
        } else {
            C xk, xlk;
            untangle<T>(a, smrow[fft_pad<E>(L - t)], TWS ? twh[t] : __ldg(&twh[t]), xk, xlk);
            if (X.act) { dst[spec_index(G, y, t)] = xk; dst[spec_index(G, y, L - t)] = xlk; }
        }
    }
    if ((TF & (G.C - 1)) == 0) {
        // TF is a multiple of the tile width: kx -> kx + TF moves TF/C tiles on, i.e. TF*ny elements
        const size_t stride = (size_t)TF * (size_t)G.ny;
        C *pa = dst + spec_index(G, y, t);
        C *pb = dst + spec_index(G, y, L - TF - t) + stride;
        C wt = mk<T>((T)1, (T)0);
        if constexpr (kRowTwc<T, E>) wt = TWS ? twh[t] : __ldg(&twh[t]);
#pragma unroll
        for (int i = 1; i < E / 2; ++i) {
            const int k = t + TF * i;
            C xk, xlk;
            C wk;
            if constexpr (kRowTwc<T, E>) wk = cmul(wt, twc_const<T, E>(i)); else wk = TWS ? twh[k] : __ldg(&twh[k]);
            untangle<T>(smrow[fft_pad<E>(k)], smrow[fft_pad<E>(L - k)], wk, xk, xlk);
            if (X.act) { pa[(size_t)i * stride] = xk; *(pb - (size_t)i * stride) = xlk; }
        }
    } else {
#pragma unroll 4
        for (int i = 1; i < E / 2; ++i) {
            const int k = t + TF * i;
            C xk, xlk;
            untangle<T>(smrow[fft_pad<E>(k)], smrow[fft_pad<E>(L - k)], TWS ? twh[k] : __ldg(&twh[k]), xk, xlk);
            if (X.act) { dst[spec_index(G, y, k)] = xk; dst[spec_index(G, y, L - k)] = xlk; }
        }
    }
}

// MK: the plan has a boundary mask (alphaR plane present); a template parameter so that the unmasked kernels carry none of
// the mask branches (their registers and instructions cost 1.2-2.3 us per row kernel at 2048^2)
template <typename T, int L, int MODE, bool MK>
__global__ void __launch_bounds__(256, SGP_ROW_MINB) row_fwd_kernel(const RowParams<T> P)
{
    using C = cx<T>;
    constexpr int E = fft_E<T>(L);
    constexpr int TF = L / E;
    constexpr int RS = row_stride(L, E);
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C *sm = reinterpret_cast<C *>(smem_raw);
    pdl_trigger();
    pdl_wait();
    RowPtrs<T> X = row_ptrs(P);                                  // this problem's arrays (batched plans: blockIdx.z)
    // the stop flag is tested only before the first store, so that its load overlaps the loads of the row
    const int stop = P.check_status ? X.ct->status : 0;

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
    C v[E];
    float accf = 0.f;
    double acc[1] = {0.0};
    constexpr bool TWS = SGP_TW_SMEM != 0;
    C *tw_s = sm + (size_t)G.RB * RS;                            // shared-memory copies of the twiddle tables, behind the rows
    if constexpr (TWS && MODE != RF_RATIO) row_tables_issue<T, L>(tw_s, P, tid, (int)blockDim.x);

    // ---- load stage with the fused elementwise work
    if constexpr (MODE == RF_PLAIN) {
        if (P.lazy == 4 && X.ct->refresh_due == 0) return;          // refresh round (A21): only after every n-th iteration
        // plain rows, optionally multiplied by M_S (input of A^T, Eq.17) or M_R (input of A, Eq.16)
        const T *src = X.in0 + (size_t)j * P.plane + (size_t)y * nx;
        const bool rowin = (unsigned)(y - G.oy) < (unsigned)G.sy;
#pragma unroll
        for (int e = 0; e < E; ++e) {
            const int x0 = 2 * (t + TF * e);
            C w2 = ld2<T>(src + x0);
            if (P.maskmode == MM_S) {
                if (!(rowin && (unsigned)(x0 - G.ox) < (unsigned)G.sx)) w2.x = (T)0;
                if (!(rowin && (unsigned)(x0 + 1 - G.ox) < (unsigned)G.sx)) w2.y = (T)0;
            } else if (P.maskmode == MM_R && MK) {
                C a2 = ld2<T>(P.alphaR + (size_t)y * nx + x0);
                if (!(a2.x > (T)0)) w2.x = (T)0;
                if (!(a2.y > (T)0)) w2.y = (T)0;
            }
            v[e] = w2;
        }
    } else if constexpr (MODE == RF_SETUP) {
        if (P.submode == RFS_PSF) {
            // K_j normalised to unit volume and circularly shifted so that its centre sits at (0,0) (A18)
            const T *src = X.in0 + (size_t)j * P.plane;
            const T inv = (T)(1.0 / X.ct->psf_sum);
            int ys = y + P.cy; if (ys >= G.ny) ys -= G.ny;
#pragma unroll
            for (int e = 0; e < E; ++e) {
                int x0 = 2 * (t + TF * e) + P.cxs; if (x0 >= nx) x0 -= nx;
                int x1 = x0 + 1; if (x1 >= nx) x1 -= nx;
                v[e] = mk<T>(src[(size_t)ys * nx + x0] * inv, src[(size_t)ys * nx + x1] * inv);
            }
        } else {   // RFS_MASK_S
#pragma unroll
            for (int e = 0; e < E; ++e) {
                int x0 = 2 * (t + TF * e);
                v[e] = mk<T>(in_S(G, y, x0) ? (T)1 : (T)0, in_S(G, y, x0 + 1) ? (T)1 : (T)0);
            }
        }
    } else if constexpr (MODE == RF_RATIO) {
        // a1: r_j = g_j / (q_j + b_j) on S (Eq.11/14/18).  In the SGP loop (lazy) the q planes are double-buffered and
        // Ctrl::need_k1 says what is left to do: 0 = nothing (the fused line-search kernel accepted lambda = 1 and has
        // already formed q(k+1), the ratio and this very spectrum), 1 = ratio of the current q (first iteration),
        // 2 = a10 after a backtrack: q(k+1) = q(k) + lambda u_j into the other buffer, then the ratio.
        const size_t base = (size_t)j * P.plane + (size_t)y * nx;
        const T bc = (T)(P.slab ? X.ct->bconst[j] : P.bconst[j]);      // batched plans: per-problem backgrounds live in the control block
        const bool rowin = (unsigned)(y - G.oy) < (unsigned)G.sy;
        int todo = 1, sel = 0;
        T lam = (T)1;
        if (P.lazy) {
            // SGP loop.  This kernel follows the line-search kernel K6.  If K6 rejected lambda = 1, the Armijo backtracking
            // (a9 for lambda < 1, elementwise on q_j + lambda u_j) runs here first, by all CTAs of the grid
            // (aux.cuh: backtrack_rounds); it ends with the book-keeping of the accepted step (finish_iteration).
            Ctrl *ct = X.ct;
            // one round trip for everything the kernel needs from the control block ...
            const int acc0 = ct->accepted;
            int st0 = ct->status, nk = ct->need_k1, qs = ct->qsel;
            double lm = ct->lambda;
            if (st0 != 0) return;
            if (P.lazy == 1 && acc0 == 0) {
                backtrack_rounds<T>(static_cast<const BtInfo<T> *>(X.btinfo));
                // ... and once more, as the accepted step left it (written by another CTA: read past the L1)
                st0 = __ldcg(&ct->status); nk = __ldcg(&ct->need_k1); qs = __ldcg(&ct->qsel); lm = __ldcg(&ct->lambda);
                if (st0 != 0) return;
            }
            todo = nk; if (todo == 0) return; sel = qs;
            lam = (T)lm;
        }
        if constexpr (TWS) row_tables_issue<T, L>(tw_s, P, tid, (int)blockDim.x);      // after the early returns above
        const bool pend = todo == 2;
        const T *qsrc = X.in1 + (size_t)(pend ? sel ^ 1 : sel) * P.qbuf;
        T *qdst = X.out0 + (size_t)sel * P.qbuf;
        // loads of a batch are issued before its stores (q is updated in place: the compiler would otherwise
        // serialise every load behind the previous store)
        constexpr int U = fwd_batch<T>(E);
#pragma unroll
        for (int e0 = 0; e0 < E; e0 += U) {
            C g2[U], q2[U], u2[U], b2[U];
            if (rowin) {
#pragma unroll
                for (int u = 0; u < U; ++u) {
                    const int x0 = 2 * (t + TF * (e0 + u));
                    g2[u] = ld2<T>(X.in0 + base + x0);
                    q2[u] = ld2<T>(qsrc + base + x0);
                    if (pend) u2[u] = ld2<T>(X.in3 + base + x0);
                    b2[u] = P.b_is_array ? ld2<T>(X.in2 + base + x0) : mk<T>(bc, bc);
                }
            }
            if (e0 == 0 && stop != 0) return;
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const int x0 = 2 * (t + TF * (e0 + u));
                C r = mk<T>((T)0, (T)0);
                if (rowin) {
                    C qn = q2[u];
                    if (pend) {
                        qn.x = qn.x + lam * u2[u].x; qn.y = qn.y + lam * u2[u].y;
                        st2_if<T>(X.act, qdst + base + x0, qn);
                    }
                    if ((unsigned)(x0 - G.ox) < (unsigned)G.sx)     r.x = ratio_term(g2[u].x, qn.x + b2[u].x);
                    if ((unsigned)(x0 + 1 - G.ox) < (unsigned)G.sx) r.y = ratio_term(g2[u].y, qn.y + b2[u].y);
                }
                v[e0 + u] = r;
            }
        }
    } else {   // RF_PROJECT
        // a4 + a7: D = (M_R/alpha) clip(f,L1,L2) (Eq.10/23); y = P+(f - alpha_k D grad) (Eq.6); d = y - f; gd = grad'd.
        // Every byte the row needs is requested before the first is used -- ONE global round trip instead of one per
        // batch (a third of this kernel's time was spent waiting at the first use of each batch): the f row goes to the
        // row's shared-memory line by cp.async (no registers), the gradient row straight into the FFT registers v[];
        // d then replaces the gradient in v[].
        const size_t base = (size_t)y * nx;
        C *frow = sm + row * RS;                                  // natural order: pair m at frow[m]
        {
            constexpr int CH = (int)(L * sizeof(C) / 16) / TF;    // 16-byte chunks per thread
            const unsigned int sdst = (unsigned int)__cvta_generic_to_shared(frow);
            const char *gsrc = reinterpret_cast<const char *>(X.in0 + base);
#pragma unroll
            for (int i = 0; i < CH; ++i) {
                const int ch = t + TF * i;
                asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(sdst + 16u * ch), "l"(gsrc + 16 * (size_t)ch) : "memory");
            }
            asm volatile("cp.async.commit_group;" ::: "memory");
        }
#pragma unroll
        for (int e = 0; e < E; ++e) v[e] = ld2<T>(X.in1 + base + 2 * (t + TF * e));
        const T alpha = (T)X.ct->alpha, L1 = (T)X.ct->L1, L2 = (T)X.ct->L2;
        const T Wc = (T)(1.0 / (double)G.p);
        // flux-constrained projection (Bonettini et al. 2009): y = max(0, x - mu D), mu from flux_mu_kernel
        const T mu = P.o.flux_constraint ? (T)X.ct->mu : (T)0;
        asm volatile("cp.async.wait_group 0;" ::: "memory");
        const SyncGroup<TFP> rsync{1 + row};
        rsync();                                                  // the copies of all threads of the row have landed
        if (stop != 0) return;
        constexpr int U = fwd_batch<T>(E);
#pragma unroll
        for (int e0 = 0; e0 < E; e0 += U) {
            C a2[U];
            if (MK) {
#pragma unroll
                for (int u = 0; u < U; ++u) a2[u] = ld2<T>(P.alphaR + base + 2 * (t + TF * (e0 + u)));
            }
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const int x0 = 2 * (t + TF * (e0 + u));
                const C f2 = frow[t + TF * (e0 + u)], g2 = v[e0 + u];
                C w2 = mk<T>(Wc, Wc);
                bool r0 = true, r1 = true;
                if (MK) {
                    r0 = a2[u].x > (T)0; r1 = a2[u].y > (T)0;
                    w2.x = r0 ? (T)1 / a2[u].x : (T)0; w2.y = r1 ? (T)1 / a2[u].y : (T)0;
                }
                C d2;
                {
                    T D = w2.x * clipT<T>(f2.x, L1, L2);
                    T yv = f2.x - alpha * D * g2.x;
                    if (P.o.flux_constraint) yv = yv - mu * D;
                    d2.x = r0 ? ((yv > (T)0 ? yv : (T)0) - f2.x) : (T)0;
                    D = w2.y * clipT<T>(f2.y, L1, L2);
                    yv = f2.y - alpha * D * g2.y;
                    if (P.o.flux_constraint) yv = yv - mu * D;
                    d2.y = r1 ? ((yv > (T)0 ? yv : (T)0) - f2.y) : (T)0;
                }
                if constexpr (sizeof(T) == 4) {
                    accf += g2.x * d2.x + g2.y * d2.y;
                    if (((e0 + u) & 3) == 3) { acc[0] += (double)accf; accf = 0.f; }
                } else {
                    acc[0] += (double)g2.x * (double)d2.x + (double)g2.y * (double)d2.y;
                }
                st2_if<T>(X.act, X.out0 + base + x0, d2);
                v[e0 + u] = d2;
            }
        }
        acc[0] += (double)accf;
        if (!act) acc[0] = 0.0;                                   // padding lanes repeat lane TF - 1: not twice in the sum
    }

    if (stop != 0) return;
    C *smrow = sm + row * RS;
    const SyncGroup<TFP> sync{1 + row};
    if constexpr (TWS) row_tables_wait();
    fwd_fft_store<T, L, TWS>(v, smrow, t, sync, P, X, y, j, TWS ? tw_s : P.tw, TWS ? tw_s + even_up(tw_total(L, E)) : P.twh);

    if constexpr (MODE == RF_PROJECT) {
        __shared__ double red[32];
        block_reduce_sum<1>(acc, red);
        if (tid == 0) X.part[blockIdx.x] = acc[0];
    }
}

}  // namespace sgpk
