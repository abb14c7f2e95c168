// small.cuh -- the whole SGP iteration (Algorithm 1) of a SMALL grid in ONE
// persistent kernel run by ONE thread-block cluster per problem ("small grids").
//
// At 256^2 / 512^2 the six launches of an iteration (row_fwd / col / row_inv kernels) are latency-bound: ~6 us each
// whatever their grid, 34-42 us per iteration for 0.26-1 Mpixel.  Here a cluster of NC CTAs keeps the problem on chip:
// CTA r owns rows [r R, (r+1) R) of the image for the row passes and columns [r CW, (r+1) CW) of the half spectrum for the
// column passes; the two transpositions of every 2-D transform go through DISTRIBUTED SHARED MEMORY (each CTA WRITES
// the pieces of its result into the shared memory of the CTAs that need them next, by asynchronous stores whose bytes
// are counted on an mbarrier of the receiving CTA: remote loads would each wait a round trip, and plain remote stores
// need a cluster barrier whose release fence waits for their acknowledgement), and the
// global sums (BB dot products, grad'd, J) are gathered in CTA 0, whose thread 0 runs the scalar logic of sgp_dev.cuh
// (bb_step, Armijo test, finish_iteration) and broadcasts the decision to every CTA's shared memory.  The planes
// (f, grad, d, q, g) stay in global memory (L1 / L2 resident: every row is only ever touched by the CTA that owns it).
// Armijo backtracks cost one reduction each: q, u, g of a row are at hand.
//
// Same arithmetic per pixel as the launch-per-pass path (ew.cuh), same FFT (fft_core.cuh), same tables and transfer
// functions; sums are grouped per CTA of this kernel, so the two paths agree to rounding, not bit for bit.
// Scope: SGP and Richardson-Lucy, one image, with or without boundary-effect correction, constant background, no replay / flux /
// refresh / Eq.25 options -- the host
// (plan_run.inl) takes the launch-per-pass path for everything else.
#pragma once
#include <cooperative_groups.h>
#include "row_inv.cuh"
#include "col.cuh"
#include "small_params.h"

namespace sgpk {

// decision of CTA 0, copied to every CTA of the cluster
struct SmallBcast {
    double alpha, lambda, L1, L2;
    int state;                        // line search: 0 = step accepted, 1 = next trial, 2 = gave up (status set)
    int status, k;
};

// elements per thread of the FFTs of this kernel: fewer than the launch-per-pass kernels use (16 / 32 in float), because a
// cluster has only NC SMs for the whole problem and the short per-thread instruction streams of 4-8 warps per scheduler hide
// each other's latencies (measured at 256^2 float: E = 16, 4 warps per SM, 43 us per iteration; E = 8: 31 us at the same stage;
// E = 4 with 16 warps adds two exchanges per transform and is no faster: 26.8 vs 25.1 us per iteration); the pass tables of these
// plans are uploaded by the host beside the plan's own (plan_impl.inl)
template <typename T> __host__ __device__ constexpr int small_E() { return 8; }

template <typename T, int NY, int NX, int NC> struct SmallCfg {
    static constexpr int L = NX / 2, Er = small_E<T>(), Ec = small_E<T>(), TFr = L / Er, TFc = NY / Ec;
    static constexpr int R = NY / NC, CW = L / NC;
    static constexpr int NTR = R * TFr, NTC = CW * TFc, NT = NTR > NTC ? NTR : NTC;
    static constexpr int SRP = L + 1;                                   // pitch of the spectrum rows (odd: the column gather spreads over the banks)
    static constexpr int RS = row_stride(L, Er), CS = (fft_padded_len(NY, Ec) + 1) & ~1;
    static constexpr int CWP = CW + 1;                                  // pitch of the column slab [ky][CWP] (the threads of a column read 32 rows at once)
    static constexpr size_t n_srow = ((size_t)R * SRP + 1) & ~(size_t)1, n_scol = ((size_t)NY * CWP + 1) & ~(size_t)1;
    static constexpr size_t n_lines = (size_t)R * RS > (size_t)CW * CS ? (size_t)R * RS : (size_t)CW * CS;
    static constexpr size_t smem = (n_srow + n_scol + n_lines) * sizeof(cx<T>);
    static constexpr bool ok = TFr <= 32 && (TFc <= 32 || CW <= 15) && R >= 1 && CW >= 1 && NT % 32 == 0 && NT <= 1024 && NTR % 32 == 0 && NTC % 32 == 0 &&
                               smem <= 200 * 1024 && plan_ok(L, Er) && plan_ok(NY, Ec);
};

// ---- asynchronous stores into the shared memory of another CTA of the cluster (st.async, sm_90+): the store is posted, and its
// bytes are counted on an mbarrier of the DESTINATION CTA, which therefore knows when a whole slab has arrived without any
// fence on the sending side (a cluster barrier with release semantics made every sender wait for the acknowledgement of its
// remote stores: "membar" was the top stall of the first versions of this kernel)
__device__ __forceinline__ unsigned int cluster_addr(const void *smem_ptr, int rank)
{
    unsigned int r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"((unsigned int)__cvta_generic_to_shared(smem_ptr)), "r"(rank));
    return r;
}
__device__ __forceinline__ void st_async(unsigned int raddr, float2 v, unsigned int rbar)
{
    const unsigned long long bits = ((unsigned long long)__float_as_uint(v.y) << 32) | (unsigned long long)__float_as_uint(v.x);
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.b64 [%0], %1, [%2];" ::"r"(raddr), "l"(bits), "r"(rbar) : "memory");
}
__device__ __forceinline__ void st_async(unsigned int raddr, double2 v, unsigned int rbar)
{
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v2.b64 [%0], {%1, %2}, [%3];"
                 ::"r"(raddr), "l"(__double_as_longlong(v.x)), "l"(__double_as_longlong(v.y)), "r"(rbar) : "memory");
}
__device__ __forceinline__ void mbar_expect(unsigned long long *bar, unsigned int bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}

__device__ __forceinline__ float kl_pair(float g0, float y0, float g1, float y1)
{
    bool ok0, ok1;
    float k0 = kl_series(g0, y0, ok0), k1 = kl_series(g1, y1, ok1);
    if (!ok0) k0 = kl_far(g0, y0);
    if (!ok1) k1 = kl_far(g1, y1);
    return k0 + k1;
}
__device__ __forceinline__ double kl_pair(double g0, double y0, double g1, double y1) { return kl_term(g0, y0) + kl_term(g1, y1); }
// the same over the pixels of the pair that lie in S (boundary-effect correction: J0 is summed over S, reading A12)
__device__ __forceinline__ float kl_pair_s(float g0, float y0, float g1, float y1, bool s0, bool s1)
{
    bool ok0, ok1;
    float k0 = kl_series(g0, y0, ok0), k1 = kl_series(g1, y1, ok1);
    if (s0 && !ok0) k0 = kl_far(g0, y0);
    if (s1 && !ok1) k1 = kl_far(g1, y1);
    return (s0 ? k0 : 0.f) + (s1 ? k1 : 0.f);
}
__device__ __forceinline__ double kl_pair_s(double g0, double y0, double g1, double y1, bool s0, bool s1)
{
    return (s0 ? kl_term(g0, y0) : 0.0) + (s1 ? kl_term(g1, y1) : 0.0);
}

// forward transform of one row held as v[e] = (x[2m], x[2m+1]), m = t + TF e; its half spectrum (entry 0 packs kx = 0 and
// nx/2) goes to dst[0 .. L-1] in shared memory (row_fwd.cuh: fwd_fft_store, with the store redirected)
template <typename T, int L, int E, typename SYNC, typename PUT>
__device__ __forceinline__ void small_fwd(cx<T> (&v)[E], cx<T> *line, const int t, const SYNC &sync, const PUT &put,
                                          const cx<T> *tw, const cx<T> *twh)
{
    using C = cx<T>;
    constexpr int TF = L / E;
    fft_block<T, L, E, -1, false>(v, line, 1, t, tw, sync);
    sync();
#pragma unroll
    for (int e = 0; e < E; ++e) line[fft_pad<E>(t + TF * e)] = v[e];
    sync();
    {
        const C a = line[fft_pad<E>(t)];
        if (t == 0) {
            put(0, mk<T>(a.x + a.y, a.x - a.y));
            put(L / 2, cconj(line[fft_pad<E>(L / 2)]));
        } else {
            C xk, xlk;
            untangle<T>(a, line[fft_pad<E>(L - t)], __ldg(&twh[t]), xk, xlk);
            put(t, xk); put(L - t, xlk);
        }
    }
#pragma unroll
    for (int i = 1; i < E / 2; ++i) {
        const int k = t + TF * i;
        C xk, xlk;
        untangle<T>(line[fft_pad<E>(k)], line[fft_pad<E>(L - k)], __ldg(&twh[k]), xk, xlk);
        put(k, xk); put(L - k, xlk);
    }
}

// MK: boundary-effect correction (Eq.16-23): S inside the grid, alphaR > 0 marks R and 1/alphaR is the weight M_R/alpha
// RL: plain Richardson-Lucy (Eq.1 / Eq.21, with the relaxations Eq.3 / Eq.4) instead of SGP: the same passes, one global sum per round
// TWO: compiled for two resident CTAs per SM (128 registers instead of 255, planes loaded where they are used): two clusters share
// the SMs of a GPC and hide each other's latencies -- the form for batches larger than the device can hold clusters of the first form
template <typename T, int NY, int NX, int NC, bool MK, bool RL, bool TWO>
__global__ void __launch_bounds__(SmallCfg<T, NY, NX, NC>::NT, TWO ? 2 : 1) small_sgp_kernel(const SmallParams<T> P)
{
    namespace cgx = cooperative_groups;
    using C = cx<T>;
    using K = SmallCfg<T, NY, NX, NC>;
    constexpr int L = K::L, Er = K::Er, Ec = K::Ec, TFr = K::TFr, TFc = K::TFc, R = K::R, CW = K::CW;
    constexpr int SRP = K::SRP, RS = K::RS, CS = K::CS, CWP = K::CWP;
    static_assert(K::Er <= 16, "the S mask of a thread's pixels is kept in 32 bits");
    static_assert(K::ok, "small_sgp_kernel: unsupported geometry");
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C *Rin = reinterpret_cast<C *>(smem_raw);                  // [R][SRP]: this CTA's spectrum rows, written by the column passes of all CTAs
    C *Cin = Rin + K::n_srow;                                  // [NY][CWP]: this CTA's spectrum columns, written by the row passes of all CTAs
    C *lines = Cin + K::n_scol;
    __shared__ double red[kNQ * 32];
    __shared__ double cpart[NC][4];
    __shared__ SmallBcast bc;
    __shared__ unsigned long long bar_c, bar_r;                // count the bytes arriving in Cin / Rin (one phase per fill)
    __shared__ C kbs[NY];                                      // companion of the packed column (CTA 0, column 0)
    __shared__ Ctrl sct;                                       // CTA 0: the control block while the kernel runs (written back at the end)

    cgx::cluster_group cluster = cgx::this_cluster();
    const int rank = (int)cluster.block_rank();
    const int pz = (int)blockIdx.x / NC;                       // problem of a batched plan
    const size_t off = (size_t)pz * P.slab, toff = (size_t)pz * P.tr_slab;
    Ctrl *ct = bshift(P.ct, off);
    T *f = bshift(P.f, off), *grad = bshift(P.grad, off), *dpl = bshift(P.d, off);
    const T *gpl = bshift(P.g, off);
    Trace tr = P.tr;
    tr.J = bshift(tr.J, toff); tr.alpha = bshift(tr.alpha, toff); tr.lambda = bshift(tr.lambda, toff);
    tr.rule = bshift(tr.rule, toff); tr.backtracks = bshift(tr.backtracks, toff);
    const DevOpts &o = P.o;

    const int tid = threadIdx.x;
    const bool ract = tid < K::NTR, cact = tid < K::NTC;
    const int row = ract ? tid / TFr : 0, t = tid % TFr;
    const int y = rank * R + row;
    const int cc = cact ? tid / TFc : 0, tc = tid % TFc;
    const int kx = rank * CW + cc;
    C *line = lines + (size_t)row * RS;                         // row passes
    C *cline = lines + (size_t)cc * CS;                         // column passes
    const C *rrow = Rin + (size_t)row * SRP;
    const SyncGroup<TFr> rsync{0};
    const SyncGroup<TFc> csync{1 + cc};                          // columns of more than 32 threads: one named barrier each
    const size_t base = (size_t)y * NX;

    // state at the start of this launch (written by the set-up kernels or by the previous launch)
    if (ct->status != 0) return;                                // uniform over the cluster
    T *q = bshift(P.q, off) + (size_t)ct->qsel * P.qbuf;
    const T bcst = (T)(P.slab ? ct->bconst[0] : P.bconst);
    const T pT = (T)1, Wc = (T)1;                               // one image without a mask: alpha = 1, W = 1 (Eq.10)
    // masks of this thread's pixels: bit 2e / 2e+1 of smask = pixel x0 / x0 + 1 of pair e lies in S; a2[e] = alpha on R, 0 outside R
    unsigned int smask = 0xffffffffu;
    C a2[MK ? Er : 1];
    if constexpr (MK) {
        smask = 0u;
        const bool rowin = (unsigned)(y - P.G.oy) < (unsigned)P.G.sy;
#pragma unroll
        for (int e = 0; e < Er; ++e) {
            const int x0 = 2 * (t + TFr * e);
            if (rowin && (unsigned)(x0 - P.G.ox) < (unsigned)P.G.sx) smask |= 1u << (2 * e);
            if (rowin && (unsigned)(x0 + 1 - P.G.ox) < (unsigned)P.G.sx) smask |= 2u << (2 * e);
            a2[e] = ract ? ld2<T>(P.alphaR + base + x0) : mk<T>((T)0, (T)0);
        }
    }
    auto in_s0 = [&](int e) -> bool { return !MK || ((smask >> (2 * e)) & 1u) != 0u; };
    auto in_s1 = [&](int e) -> bool { return !MK || ((smask >> (2 * e + 1)) & 1u) != 0u; };
    // ratio g / (q + b) on S, 0 elsewhere (Eq.18)
    auto ratio_pair = [&](int e, const C g2_, const C q2_) -> C {
        return mk<T>(in_s0(e) ? ratio_term(g2_.x, q2_.x + bcst) : (T)0, in_s1(e) ? ratio_term(g2_.y, q2_.y + bcst) : (T)0);
    };
    if (tid == 0) {
        sct = *ct;                                              // every CTA keeps its own replica of the control block (see decide below)
        bc.alpha = sct.alpha; bc.lambda = sct.lambda; bc.L1 = sct.L1; bc.L2 = sct.L2; bc.state = 0; bc.status = 0; bc.k = sct.k;
    }
    __syncthreads();
    Ctrl *const gct = ct;
    ct = &sct;                                                  // used by thread 0 only from here on
    // Global sums without a second barrier: every CTA sends its partial sums to ALL CTAs of the cluster; after ONE cluster
    // barrier thread 0 of every CTA adds the NC partials in the same order and runs the same scalar logic (bb_step, Armijo
    // test, finish_iteration) on its own replica of the control block -- identical inputs, identical decisions.  Only CTA 0
    // writes the traces and, at the end, the control block itself.
    if (rank != 0) { tr.J = nullptr; tr.alpha = nullptr; tr.lambda = nullptr; tr.rule = nullptr; tr.backtracks = nullptr; }
    __shared__ double mypart[4];
    auto send_partials = [&](const double *vals, int nq) {     // vals: valid in thread 0 (block_reduce_sum)
        if (tid == 0) for (int i = 0; i < nq; ++i) mypart[i] = vals[i];
        __syncthreads();
        if (tid < NC) {
            double *dst = cluster.map_shared_rank(&cpart[0][0], tid) + rank * 4;
            for (int i = 0; i < nq; ++i) dst[i] = mypart[i];
        }
    };

    // half-spectrum entry k of this thread's row -> the column slab of the CTA that owns column k
    const unsigned int cin_u = (unsigned int)__cvta_generic_to_shared(Cin), rin_u = (unsigned int)__cvta_generic_to_shared(Rin);
    const unsigned int barc_u = smem_u32(&bar_c), barr_u = smem_u32(&bar_r);
    auto rmap = [&](unsigned int a, int r) -> unsigned int { unsigned int o_; asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(o_) : "r"(a), "r"(r)); return o_; };
    auto put_row = [&](const int k, const C val) {
        const int dst = k / CW;
        st_async(rmap(cin_u + (unsigned int)(((size_t)y * CWP + (k % CW)) * sizeof(C)), dst), val, rmap(barc_u, dst));
    };
    constexpr unsigned int CIN_BYTES = (unsigned int)((size_t)NY * CW * sizeof(C)), RIN_BYTES = (unsigned int)((size_t)R * L * sizeof(C));
    unsigned int ph_c = 0, ph_r = 0;
    // all of Cin / Rin has arrived (thread 0 arms the phase: one arrival + the slab's bytes), and no thread of this CTA is still in the previous pass
    auto wait_cin = [&](void) { if (tid == 0) mbar_expect(&bar_c, CIN_BYTES); mbar_wait(&bar_c, ph_c); ph_c ^= 1; __syncthreads(); };
    auto wait_rin = [&](void) { if (tid == 0) mbar_expect(&bar_r, RIN_BYTES); mbar_wait(&bar_r, ph_r); ph_r ^= 1; __syncthreads(); };
    // the transfer function of this thread's column entries stays in registers for the whole run (it is read twice per iteration)
    C kh[Ec];
    if (cact) {
#pragma unroll
        for (int e = 0; e < Ec; ++e) kh[e] = __ldg(&P.khat[spec_index(P.G, tc + TFc * e, kx)]);
    }
    if (rank == 0) for (int i = tid; i < NY; i += K::NT) kbs[i] = __ldg(&P.khatB[i]);
    __syncthreads();
    C v[Er > Ec ? Er : Ec];
#ifdef SGP_SMALL_TIMING
    int dbg_n = 0;
#define SMALL_TICK() do { if (P.dbg && rank == 0 && tid == 0 && dbg_it && dbg_n < 64) { unsigned long long t_; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_)); P.dbg[dbg_n++] = t_; } } while (0)
#else
#define SMALL_TICK() do { } while (0)
#endif

    // ---- a1: r = g / (q + b) for this CTA's rows, forward row transform -> the column slabs of all CTAs
    auto ratio_rows = [&](void) {
        if (ract) {
            C (&vr)[Er] = reinterpret_cast<C (&)[Er]>(v);
#pragma unroll
            for (int e = 0; e < Er; ++e) {
                const int x0 = 2 * (t + TFr * e);
                const C g2 = ld2<T>(gpl + base + x0), q2 = ld2<T>(q + base + x0);
                vr[e] = ratio_pair(e, g2, q2);
            }
            small_fwd<T, L, Er>(vr, line, t, rsync, put_row, P.tw_r, P.tw_h);
        }
    };

    // ---- a2 / a8: column pass of this CTA's columns (all of Cin has arrived): forward FFT, x conj(K^) or x K^, inverse FFT; entry
    //      (ky, kx) of the result goes to the row buffer of the CTA that owns row ky
    auto col_pass = [&](const bool conj) {
        if (cact) {
            C (&vc)[Ec] = reinterpret_cast<C (&)[Ec]>(v);
#pragma unroll
            for (int e = 0; e < Ec; ++e) vc[e] = Cin[(size_t)(tc + TFc * e) * CWP + cc];
            fft_block<T, NY, Ec, -1, false>(vc, cline, 1, tc, P.tw_c, csync);
            // the packed column (kx = 0 holds kx = 0 and nx/2, col.cuh) needs its own reflection C~[ky] = conj C[-ky]: every column
            // parks its transform in its line (the threads of several columns may share a warp and must stay in step)
            csync();
#pragma unroll
            for (int e = 0; e < Ec; ++e) cline[fft_pad<Ec>(tc + TFc * e)] = vc[e];
            csync();
#pragma unroll
            for (int e = 0; e < Ec; ++e) vc[e] = conj ? cmulc(vc[e], kh[e]) : cmul(vc[e], kh[e]);
            if (kx == 0) {
#pragma unroll
                for (int e = 0; e < Ec; ++e) {
                    const int ky = tc + TFc * e, kyn = ky == 0 ? 0 : NY - ky;
                    const C ctl = cconj(cline[fft_pad<Ec>(kyn)]);
                    vc[e] = cadd(vc[e], conj ? cmulc(ctl, kbs[ky]) : cmul(ctl, kbs[ky]));
                }
            }
            fft_block<T, NY, Ec, +1, false>(vc, cline, 1, tc, P.tw_c, csync);
#pragma unroll
            for (int e = 0; e < Ec; ++e) {
                const int ky = tc + TFc * e, dst = ky / R;
                st_async(rmap(rin_u + (unsigned int)(((size_t)(ky % R) * SRP + kx) * sizeof(C)), dst), vc[e], rmap(barr_u, dst));
            }
        }
    };

    // ---- inverse row pass of this CTA's rows (all of Rin has arrived): re-tangle, inverse FFT: v[e] = (w(2m), w(2m+1))
    auto inv_rows = [&](void) {
        if (ract) {
            C (&vr)[Er] = reinterpret_cast<C (&)[Er]>(v);
            auto X = [&](int k) -> C { return rrow[k]; };
            {
                const C a = X(t);
                if (t == 0) {
                    line[0] = mk<T>(a.x + a.y, a.x - a.y);
                    const C m = X(L / 2);
                    line[fft_pad<Er>(L / 2)] = mk<T>((T)2 * m.x, (T)-2 * m.y);
                } else {
                    C zk, zlk;
                    retangle<T>(a, X(L - t), __ldg(&P.tw_h[t]), zk, zlk);
                    line[fft_pad<Er>(t)] = zk; line[fft_pad<Er>(L - t)] = zlk;
                }
            }
#pragma unroll
            for (int i = 1; i < Er / 2; ++i) {
                const int k = t + TFr * i;
                C zk, zlk;
                retangle<T>(X(k), X(L - k), __ldg(&P.tw_h[k]), zk, zlk);
                line[fft_pad<Er>(k)] = zk; line[fft_pad<Er>(L - k)] = zlk;
            }
            rsync();
#pragma unroll
            for (int e = 0; e < Er; ++e) vr[e] = line[fft_pad<Er>(t + TFr * e)];
            fft_block<T, L, Er, +1, false>(vr, line, 1, t, P.tw_r, rsync);
        }
    };

    // planes of this thread's pixels.  PF (float): they are requested BEFORE the transform whose epilogue needs them and stay in
    // registers while they are valid (f from the gradient step to the update, d from the projection, g and q from the line
    // search); double: loaded where they are used (twice the registers).
    constexpr bool PF = sizeof(T) == 4 && !TWO;
    C f2[Er], d2[Er], o2[Er], g2[Er], q2[Er];
    auto ldrow = [&](C (&a)[Er], const T *plane) {
#pragma unroll
        for (int e = 0; e < Er; ++e) a[e] = ld2<T>(plane + base + 2 * (t + TFr * e));
    };
    C (&vr)[Er] = reinterpret_cast<C (&)[Er]>(v);
    // J(lambda) = sum_S kl(g, q + lambda u + b) over this CTA's rows, u in v[] (Alg.1 step 5; each trial is elementwise)
    auto eval_J = [&](const T lam) -> double {
        double acc = 0.0;
        if (ract) {
#pragma unroll
            for (int e = 0; e < Er; ++e) {
                const T y0 = (T)(q2[e].x + lam * vr[e].x) + bcst, y1 = (T)(q2[e].y + lam * vr[e].y) + bcst;
                if constexpr (MK) acc += (double)kl_pair_s(g2[e].x, y0, g2[e].y, y1, in_s0(e), in_s1(e));
                else acc += (double)kl_pair(g2[e].x, y0, g2[e].y, y1);
            }
        }
        return acc;
    };
    // thread 0 of every CTA: sum of column i of the partials, in rank order
    auto total = [&](int i) -> double { double a = 0.0; for (int r = 0; r < NC; ++r) a += cpart[r][i]; return a; };

    if (tid == 0) {
        mbar_init(&bar_c, 1); mbar_init(&bar_r, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    cluster.sync();                                             // every CTA's barriers exist before anybody sends
    if constexpr (RL) {
        // ---- a12: round k = J0(f(k)), the stopping rules, and unless one fires f(k+1) = (M_R/alpha) o f o A^T(g / (A f + b)) (Eq.1 / Eq.21).
        //      One cluster barrier per round (the sum of J0); the mbarriers of the four transposes order the re-use of the slabs.
        const T rx = (T)o.rl_relax, lamr = (T)o.rl_linear;
        const bool relax = o.rl_relax != 1.0, lin = o.rl_linear != 1.0;
        if (ract) {
            ldrow(f2, f);
#pragma unroll
            for (int e = 0; e < Er; ++e) vr[e] = f2[e];
            small_fwd<T, L, Er>(vr, line, t, rsync, put_row, P.tw_r, P.tw_h);
        }
        for (int it = 0; it < P.iters; ++it) {
            wait_cin();
            col_pass(false);                                    // A f (Eq.16)
            wait_rin();
            if (ract) ldrow(g2, gpl);
            inv_rows();                                         // v[] = A f on this CTA's rows
            {
                double pr[1] = {0.0};
                if (ract) {
#pragma unroll
                    for (int e = 0; e < Er; ++e) {
                        if (!in_s0(e)) vr[e].x = (T)0;
                        if (!in_s1(e)) vr[e].y = (T)0;
                        const T y0 = vr[e].x + bcst, y1 = vr[e].y + bcst;
                        if constexpr (MK) pr[0] += (double)kl_pair_s(g2[e].x, y0, g2[e].y, y1, in_s0(e), in_s1(e));
                        else pr[0] += (double)kl_pair(g2[e].x, y0, g2[e].y, y1);
                    }
                }
                block_reduce_sum<1>(pr, red);
                send_partials(pr, 1);
            }
            cluster.sync();
            if (tid == 0) {                                     // J0(f(k)) and the stopping rules before the k-th update (row_inv.cuh: QJ_RL)
                const double J = total(0);
                const int k = ct->k;
                const double Jold = ct->J;
                ct->J = J;
                if (tr.J) tr.J[k] = J;
                ct->nfft += 2ULL;
                if (!isfinite(J)) ct->status = SGP_ERR_NONFINITE;
                else { const int r = stop_test(o, k, J, Jold, k > 0); if (r) ct->status = r; else ct->k = k + 1; }
                bc.status = ct->status;
            }
            __syncthreads();
            if (bc.status != 0) break;
            if (ract) {
#pragma unroll
                for (int e = 0; e < Er; ++e) vr[e] = ratio_pair(e, g2[e], vr[e]);
                small_fwd<T, L, Er>(vr, line, t, rsync, put_row, P.tw_r, P.tw_h);
            }
            wait_cin();
            col_pass(true);                                     // A^T r (Eq.17)
            wait_rin();
            if (ract && !PF) ldrow(f2, f);
            inv_rows();
            const bool more = it + 1 < P.iters;
            if (ract) {
#pragma unroll
                for (int e = 0; e < Er; ++e) {
                    const T fa[2] = {f2[e].x, f2[e].y}, wa[2] = {vr[e].x, vr[e].y};
                    T ya[2];
#pragma unroll
                    for (int c = 0; c < 2; ++c) {
                        T wv = Wc;
                        if constexpr (MK) { const T av = c == 0 ? a2[e].x : a2[e].y; wv = av > (T)0 ? (T)1 / av : (T)0; }
                        ya[c] = wv * fa[c] * wa[c];
                        if (relax) ya[c] = fa[c] * pow(fmax(wv * wa[c], (T)0), rx);                              // Eq.3
                        if (lin) ya[c] = fmax(fa[c] - lamr * (fa[c] * ((T)1 - wv * wa[c])), (T)0);              // Eq.4, projected on f >= 0 (A25)
                    }
                    const C yn = mk<T>(ya[0], ya[1]);
                    st2<T>(f + base + 2 * (t + TFr * e), yn);
                    f2[e] = yn; vr[e] = yn;
                }
                if (more) small_fwd<T, L, Er>(vr, line, t, rsync, put_row, P.tw_r, P.tw_h);
            }
            if (tid == 0) ct->nfft += 2ULL;
            if (!more) break;
        }
        if (rank == 0 && tid == 0) *gct = sct;
        return;
    }
    ratio_rows();
    double gd_part = 0.0, Jref = 0.0, gdt = 0.0;
    for (int it = 0; it < P.iters; ++it) {
#ifdef SGP_SMALL_TIMING
        const bool dbg_it = it == 5;
#endif
        SMALL_TICK();
        wait_cin();
        SMALL_TICK();
        col_pass(true);                                         // a2: A^T r in Fourier space (Eq.17)
        SMALL_TICK();
        wait_rin();
        SMALL_TICK();
        const int k = bc.k;
        if (ract && PF) { ldrow(f2, f); if (k > 0) { ldrow(d2, dpl); ldrow(o2, grad); } }
        inv_rows();
        // ---- a3 + a5: grad = 1 - w; BB sums with s = lambda d, z = grad - grad_prev, D = clip(f, L1, L2) (Eq.7-8, Eq.10)
        {
            const T lam = (T)bc.lambda, L1 = (T)bc.L1, L2 = (T)bc.L2;
            double acc[4] = {0.0, 0.0, 0.0, 0.0};
            if (ract) {
                if (!PF && k > 0) { ldrow(f2, f); ldrow(d2, dpl); ldrow(o2, grad); }
#pragma unroll
                for (int e = 0; e < Er; ++e) {
                    C gn = mk<T>(pT - vr[e].x, pT - vr[e].y);
                    bool inR[2] = {true, true};
                    T wv[2] = {Wc, Wc};
                    if constexpr (MK) {
                        inR[0] = a2[e].x > (T)0; inR[1] = a2[e].y > (T)0;
                        wv[0] = inR[0] ? (T)1 / a2[e].x : (T)0; wv[1] = inR[1] ? (T)1 / a2[e].y : (T)0;
                        gn = mk<T>(inR[0] ? a2[e].x - vr[e].x : (T)0, inR[1] ? a2[e].y - vr[e].y : (T)0);
                    }
                    if (k > 0) {
                        const T fa[2] = {f2[e].x, f2[e].y}, da[2] = {d2[e].x, d2[e].y}, ga[2] = {gn.x, gn.y}, oa[2] = {o2[e].x, o2[e].y};
                        T pq[4] = {(T)0, (T)0, (T)0, (T)0};
#pragma unroll
                        for (int c = 0; c < 2; ++c) {
                            const T s = lam * da[c];
                            const T Di = wv[c] * clipT<T>(fa[c], L1, L2);
                            const T zr = ga[c] - oa[c];
                            const T zf = inR[c] ? zr : (T)0;
                            const T si = inR[c] ? fast_div(s, Di) : (T)0, zd = inR[c] ? zr * Di : (T)0;
                            if constexpr (sizeof(T) == 8) {
                                acc[0] += si * si; acc[1] += si * zf; acc[2] += s * zd; acc[3] += zd * zd;
                            } else {
                                pq[0] = fmaf(si, si, pq[0]); pq[1] = fmaf(si, zf, pq[1]); pq[2] = fmaf(s, zd, pq[2]); pq[3] = fmaf(zd, zd, pq[3]);
                            }
                        }
                        if constexpr (sizeof(T) == 4) {
#pragma unroll
                            for (int k4 = 0; k4 < 4; ++k4) acc[k4] += (double)pq[k4];
                        }
                    }
                    vr[e] = gn;                                 // the gradient stays in the registers for the projection
                }
            }
            block_reduce_sum<4>(acc, red);
            send_partials(acc, 4);
        }
        SMALL_TICK();
        {
            // the gradient goes to global memory between the two halves of the barrier: stored before it, the barrier's release
            // fence would wait for the acknowledgement of these (CTA-private) stores
            auto token = cluster.barrier_arrive();
            if (ract) {
#pragma unroll
                for (int e = 0; e < Er; ++e) st2<T>(grad + base + 2 * (t + TFr * e), vr[e]);
            }
            cluster.barrier_wait(std::move(token));
        }
        SMALL_TICK();
        if (tid == 0) {                                         // a6: step length, in every CTA
            const double s0 = total(0), s1 = total(1), s2 = total(2), s3 = total(3);
            bb_step(ct, o, tr, s0, s1, s2, s3);
            bc.alpha = ct->alpha;
        }
        __syncthreads();
        SMALL_TICK();
        SMALL_TICK();
        SMALL_TICK();
        // ---- a4 + a7: D = clip(f, L1, L2); y = max(0, f - alpha D grad) (Eq.6); d = y - f; grad'd; forward row transform of d
        gd_part = 0.0;
        if (ract) {
            const T alpha = (T)bc.alpha, L1 = (T)bc.L1, L2 = (T)bc.L2;
            float accf = 0.f;
            if (!PF) ldrow(f2, f);
#pragma unroll
            for (int e = 0; e < Er; ++e) {
                const C fe = f2[e], ge = vr[e];
                C de;
                bool r0 = true, r1 = true;
                T w0 = Wc, w1 = Wc;
                if constexpr (MK) {
                    r0 = a2[e].x > (T)0; r1 = a2[e].y > (T)0;
                    w0 = r0 ? (T)1 / a2[e].x : (T)0; w1 = r1 ? (T)1 / a2[e].y : (T)0;
                }
                T D = w0 * clipT<T>(fe.x, L1, L2);
                T yv = fe.x - alpha * D * ge.x;
                de.x = r0 ? ((yv > (T)0 ? yv : (T)0) - fe.x) : (T)0;
                D = w1 * clipT<T>(fe.y, L1, L2);
                yv = fe.y - alpha * D * ge.y;
                de.y = r1 ? ((yv > (T)0 ? yv : (T)0) - fe.y) : (T)0;
                if constexpr (sizeof(T) == 4) {
                    accf += ge.x * de.x + ge.y * de.y;
                    if ((e & 3) == 3) { gd_part += (double)accf; accf = 0.f; }
                } else {
                    gd_part += (double)ge.x * (double)de.x + (double)ge.y * (double)de.y;
                }
                st2<T>(dpl + base + 2 * (t + TFr * e), de);
                vr[e] = de;
                if (PF) d2[e] = de;
            }
            gd_part += (double)accf;
            small_fwd<T, L, Er>(vr, line, t, rsync, put_row, P.tw_r, P.tw_h);
        }
        SMALL_TICK();
        wait_cin();
        SMALL_TICK();
        col_pass(false);                                        // a8: A d (Eq.16)
        SMALL_TICK();
        wait_rin();
        SMALL_TICK();
        if (ract && PF) { ldrow(g2, gpl); ldrow(q2, q); }
        inv_rows();                                             // v[] = u = A d on this CTA's rows
        if constexpr (MK) {                                     // u = M_S o (...) (Eq.16): q stays zero outside S
            if (ract) {
#pragma unroll
                for (int e = 0; e < Er; ++e) { if (!in_s0(e)) vr[e].x = (T)0; if (!in_s1(e)) vr[e].y = (T)0; }
            }
        }
        if (ract && !PF) { ldrow(g2, gpl); ldrow(q2, q); }
        // ---- a9: Armijo rule, lambda = 1, theta, theta^2, ...; every trial is one reduction
        {
            double pr[2] = {eval_J((T)1), gd_part};
            block_reduce_sum<2>(pr, red);
            send_partials(pr, 2);
        }
        SMALL_TICK();
        cluster.sync();
        SMALL_TICK();
        if (tid == 0) {
            const double J = total(0);
            gdt = total(1);
            Jref = armijo_ref(ct);
            ct->gd = gdt; ct->Jref = Jref; ct->Jtrial = J;
            if (isfinite(J) && J <= Jref + o.beta * gdt) {      // Alg.1 step 5 at lambda = 1
                finish_iteration(ct, o, tr, 1.0, J, 0, 1);
                bc.state = 0; bc.lambda = 1.0;
            } else if (o.max_backtracks < 1) { ct->status = SGP_ERR_LINESEARCH; bc.state = 2; }      // A16
            else bc.state = 1;
            bc.status = ct->status; bc.k = ct->k;
        }
        __syncthreads();
        SMALL_TICK();
        SMALL_TICK();
        SMALL_TICK();
        int trial = 0;
        while (bc.state == 1) {
            double lambda = 1.0;
            for (int i = 0; i <= trial; ++i) lambda *= o.theta;               // PAPER.md:124, the oracle's own sequence of products
            double pr[1] = {eval_J((T)lambda)};
            cluster.sync();                                     // every CTA has read the partials of the previous trial
            block_reduce_sum<1>(pr, red);
            send_partials(pr, 1);
            cluster.sync();
            if (tid == 0) {
                const double Jn = total(0);
                const int nbt = trial + 1;
                if (isfinite(Jn) && Jn <= Jref + o.beta * lambda * gdt) {
                    finish_iteration(ct, o, tr, lambda, Jn, nbt, 1);
                    bc.state = 0; bc.lambda = lambda;
                } else if (nbt >= o.max_backtracks) { ct->status = SGP_ERR_LINESEARCH; bc.state = 2; }   // A16
                bc.status = ct->status; bc.k = ct->k;
            }
            __syncthreads();
            ++trial;
        }
        if (bc.state != 0) break;                               // line search gave up: f stays f(k)
        // ---- a10: f <- f + lambda d, q <- q + lambda u; then a1 of the next iteration from the new q
        const bool more = bc.status == 0 && it + 1 < P.iters;
        if (ract) {
            const T lam = (T)bc.lambda;
            if (!PF) { ldrow(f2, f); ldrow(d2, dpl); }
#pragma unroll
            for (int e = 0; e < Er; ++e) {
                const int x0 = 2 * (t + TFr * e);
                C qn, fn;
                qn.x = q2[e].x + lam * vr[e].x; qn.y = q2[e].y + lam * vr[e].y;
                fn.x = f2[e].x + lam * d2[e].x; fn.y = f2[e].y + lam * d2[e].y;
                st2<T>(q + base + x0, qn);
                st2<T>(f + base + x0, fn);
                vr[e] = ratio_pair(e, g2[e], qn);
            }
            if (more) small_fwd<T, L, Er>(vr, line, t, rsync, put_row, P.tw_r, P.tw_h);
        }
        if (tid == 0) {
            // finish_iteration keeps the books of the launch-per-pass path (lazy update, double-buffered q): here the step
            // has been applied and q updated in place.  Two 2-D transforms per operator application (n_fft2).
            ct->pending = 0; ct->qsel ^= 1; ct->nfft += 4ULL;
        }
        SMALL_TICK();
        if (!more) break;
    }
    if (rank == 0 && tid == 0) *gct = sct;
}

}  // namespace sgpk
