// row_fwd.cuh -- real rows -> half spectrum (row pass of FFT2), with the elementwise work of the iteration
// fused into the load stage.
//
// One row is transformed by TF = L/E threads (a warp for the 2048-wide grid: L = 1024, E = 32, passes 32 x 32);
// the threads of a row synchronise only among themselves (SyncGroup), so the rows of a CTA drift apart and
// the loads of one row overlap the butterflies and stores of another.  grid = (ny/RB, images), block = RB*TF
// threads, dynamic smem = RB * padded(L) complex.
#pragma once
#include "ew.cuh"

namespace sgpk {

// pairs loaded ahead of the first store of a batch in the load stage
template <typename T> __host__ __device__ constexpr int fwd_batch(int E)
{
    return sizeof(T) == 8 ? (E % 4 == 0 ? 4 : 2) : (E % 8 == 0 ? 8 : 4);
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
template <typename T, int L, typename SYNC>
__device__ __forceinline__ void fwd_fft_store(cx<T> (&v)[fft_E<T>(L)], cx<T> *smrow, const int t, const SYNC &sync,
                                              const RowParams<T> &P, const int y, const int j)
{
    using C = cx<T>;
    constexpr int E = fft_E<T>(L);
    constexpr int TF = L / E;
    const Geom &G = P.G;
    // ---- complex FFT of length L = nx/2 over z[m] = x[2m] + i x[2m+1]
    fft_block<T, L, E, -1>(v, smrow, 1, t, P.tw, sync);
    sync();
#pragma unroll
    for (int e = 0; e < E; ++e) smrow[fft_pad<E>(t + TF * e)] = v[e];
    sync();

    // ---- untangle the two interleaved real transforms, one (k, L-k) pair per step, and store tile-major:
    //      E = (Z[k] + conj Z[L-k])/2, O = -i (Z[k] - conj Z[L-k])/2, w = exp(-2 pi i k/nx):
    //      X[k] = E + w O,  X[L-k] = conj(E - w O);  entry 0 = (X[0], X[L]) packed;  X[L/2] = conj Z[L/2]
    C *dst = P.spec + (size_t)j * P.specplane;
    {   // i = 0
        const C a = smrow[fft_pad<E>(t)];
        if (t == 0) {
            dst[spec_index(G, y, 0)] = mk<T>(a.x + a.y, a.x - a.y);
            dst[spec_index(G, y, L / 2)] = cconj(smrow[fft_pad<E>(L / 2)]);
        } else {
            C xk, xlk;
            untangle<T>(a, smrow[fft_pad<E>(L - t)], __ldg(&P.twh[t]), xk, xlk);
            dst[spec_index(G, y, t)] = xk;
            dst[spec_index(G, y, L - t)] = xlk;
        }
    }
    if ((TF & (G.C - 1)) == 0) {
        // TF is a multiple of the tile width: kx -> kx + TF moves TF/C tiles on, i.e. TF*ny elements
        const size_t stride = (size_t)TF * (size_t)G.ny;
        C *pa = dst + spec_index(G, y, t);
        C *pb = dst + spec_index(G, y, L - TF - t) + stride;
#pragma unroll
        for (int i = 1; i < E / 2; ++i) {
            const int k = t + TF * i;
            C xk, xlk;
            untangle<T>(smrow[fft_pad<E>(k)], smrow[fft_pad<E>(L - k)], __ldg(&P.twh[k]), xk, xlk);
            pa[(size_t)i * stride] = xk;
            *(pb - (size_t)i * stride) = xlk;
        }
    } else {
#pragma unroll 4
        for (int i = 1; i < E / 2; ++i) {
            const int k = t + TF * i;
            C xk, xlk;
            untangle<T>(smrow[fft_pad<E>(k)], smrow[fft_pad<E>(L - k)], __ldg(&P.twh[k]), xk, xlk);
            dst[spec_index(G, y, k)] = xk;
            dst[spec_index(G, y, L - k)] = xlk;
        }
    }
}

// MK: the plan has a boundary mask (alphaR plane present); a template parameter so that the unmasked kernels carry none of
// the mask branches (their registers and instructions cost 1.2-2.3 us per row kernel at 2048^2)
template <typename T, int L, int MODE, bool MK>
__global__ void __launch_bounds__(256, 2) row_fwd_kernel(const RowParams<T> P)
{
    using C = cx<T>;
    constexpr int E = fft_E<T>(L);
    constexpr int TF = L / E;
    constexpr int RS = fft_padded_len(L, E);
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C *sm = reinterpret_cast<C *>(smem_raw);
    pdl_trigger();
    pdl_wait();
    // the stop flag is tested only before the first store, so that its load overlaps the loads of the row
    const int stop = P.check_status ? P.ct->status : 0;

    const Geom &G = P.G;
    const int tid = threadIdx.x;
    const int row = tid / TF, t = tid - row * TF;
    const int y = blockIdx.x * G.RB + row;
    const int j = blockIdx.y;
    constexpr int nx = 2 * L;
    C v[E];
    float accf = 0.f;
    double acc[1] = {0.0};

    // ---- load stage with the fused elementwise work
    if constexpr (MODE == RF_PLAIN) {
        // plain rows, optionally multiplied by M_S (input of A^T, Eq.17) or M_R (input of A, Eq.16)
        const T *src = P.in0 + (size_t)j * P.plane + (size_t)y * nx;
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
            const T *src = P.in0 + (size_t)j * P.plane;
            const T inv = (T)(1.0 / P.ct->psf_sum);
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
        const T bc = (T)P.bconst[j];
        const bool rowin = (unsigned)(y - G.oy) < (unsigned)G.sy;
        int todo = 1, sel = 0;
        if (P.lazy) {
            // Two instances of this kernel follow the line-search kernel (plan_run.inl): lazy = 1 runs BESIDE the
            // backtracking kernel and works only if lambda = 1 was accepted (Ctrl::accepted is written by the line-search
            // kernel alone, so it is stable here; nothing else of the control block is read before this test, because the
            // backtracking kernel rewrites it when it has work); lazy = 2 runs BEHIND the backtracking kernel and works
            // only if that had to find lambda < 1; lazy = 3 (plain stream order) takes either case.
            const int acc = P.ct->accepted;
            if ((P.lazy == 1 && acc == 0) || (P.lazy == 2 && acc != 0)) return;
            if (P.ct->status != 0) return;
            todo = P.ct->need_k1; if (todo == 0) return; sel = P.ct->qsel;
        }
        const bool pend = todo == 2;
        const T *qsrc = P.in1 + (size_t)(pend ? sel ^ 1 : sel) * P.qbuf;
        T *qdst = P.out0 + (size_t)sel * P.qbuf;
        const T lam = (T)P.ct->lambda;
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
                    g2[u] = ld2<T>(P.in0 + base + x0);
                    q2[u] = ld2<T>(qsrc + base + x0);
                    if (pend) u2[u] = ld2<T>(P.in3 + base + x0);
                    b2[u] = P.b_is_array ? ld2<T>(P.in2 + base + x0) : mk<T>(bc, bc);
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
                        st2<T>(qdst + base + x0, qn);
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
            const char *gsrc = reinterpret_cast<const char *>(P.in0 + base);
#pragma unroll
            for (int i = 0; i < CH; ++i) {
                const int ch = t + TF * i;
                asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(sdst + 16u * ch), "l"(gsrc + 16 * (size_t)ch) : "memory");
            }
            asm volatile("cp.async.commit_group;" ::: "memory");
        }
#pragma unroll
        for (int e = 0; e < E; ++e) v[e] = ld2<T>(P.in1 + base + 2 * (t + TF * e));
        const T alpha = (T)P.ct->alpha, L1 = (T)P.ct->L1, L2 = (T)P.ct->L2;
        const T Wc = (T)(1.0 / (double)G.p);
        asm volatile("cp.async.wait_group 0;" ::: "memory");
        const SyncGroup<TF> rsync{1 + row};
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
                    d2.x = r0 ? ((yv > (T)0 ? yv : (T)0) - f2.x) : (T)0;
                    D = w2.y * clipT<T>(f2.y, L1, L2);
                    yv = f2.y - alpha * D * g2.y;
                    d2.y = r1 ? ((yv > (T)0 ? yv : (T)0) - f2.y) : (T)0;
                }
                if constexpr (sizeof(T) == 4) {
                    accf += g2.x * d2.x + g2.y * d2.y;
                    if (((e0 + u) & 3) == 3) { acc[0] += (double)accf; accf = 0.f; }
                } else {
                    acc[0] += (double)g2.x * (double)d2.x + (double)g2.y * (double)d2.y;
                }
                st2<T>(P.out0 + base + x0, d2);
                v[e0 + u] = d2;
            }
        }
        acc[0] += (double)accf;
    }

    if (stop != 0) return;
    C *smrow = sm + row * RS;
    const SyncGroup<TF> sync{1 + row};
    fwd_fft_store<T, L>(v, smrow, t, sync, P, y, j);

    if constexpr (MODE == RF_PROJECT) {
        __shared__ double red[32];
        block_reduce_sum<1>(acc, red);
        if (tid == 0) P.part[blockIdx.x] = acc[0];
    }
}

}  // namespace sgpk
