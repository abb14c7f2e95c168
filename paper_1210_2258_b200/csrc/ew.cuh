// ew.cuh -- parameter blocks of the hot-path kernels and the per-pixel arithmetic of the SGP / RL iteration
// (DESIGN.md section 5).
//
// Data layout.  Real planes are row-major ny x nx.  A half spectrum of a real plane holds nx/2 complex
// numbers per row: entry kx = 1..nx/2-1 is the DFT coefficient, entry 0 packs the two real coefficients
// (kx = 0, kx = nx/2) as (re, im).  Spectra are stored COLUMN-TILE-MAJOR: tile = kx / C, and inside a tile
// element (ky, kx % C) sits at ky*C + kx%C, so a CTA of the column kernel reads one contiguous chunk of
// ny*C complex numbers.
#pragma once
#include <cooperative_groups.h>
#include <type_traits>
#include "fft_core.cuh"
#include "sgp_dev.cuh"

namespace sgpk {
namespace cg = cooperative_groups;

enum RowFwdMode { RF_PLAIN = 0, RF_SETUP = 1, RF_RATIO = 2, RF_PROJECT = 3, RF_NMODES = 4 };
enum RowFwdSetup { RFS_PSF = 0, RFS_MASK_S = 1 };
enum RowInvMode { RI_PLAIN = 0, RI_GRAD = 1, RI_LS = 2, RI_QJ = 3, RI_RLUPDATE = 4, RI_LSF = 5, RI_QJF = 6, RI_RLUPF = 7, RI_NMODES = 8 };
enum RowInvPlain { RIP_STORE = 0, RIP_RLMINMAX = 1, RIP_STORE_POS = 2 };
enum MaskMode { MM_NONE = 0, MM_S = 1, MM_R = 2 };
enum QJSub { QJ_INIT = 0, QJ_RL = 1, QJ_PLAIN = 2, QJ_REFRESH = 3 };
enum Ticket { TK_GRAD = 0, TK_LS = 1, TK_QJ = 2, TK_MINMAX = 3, TK_BACKTRACK = 4, TK_ERR = 5 };

template <typename T> struct RowParams {
    Geom G;
    DevOpts o;
    Trace tr;
    Ctrl *ct;
    int submode, maskmode, b_is_array;
    int lazy;                         // 1: SGP loop -- apply the pending update f += lambda d, q_j += lambda u_j on the fly
    const T *in0, *in1, *in2, *in3;   // real planes; image j at + j*plane
    T *out0, *out1;
    cx<T> *spec;                      // spectrum of image j at + j*specplane
    size_t plane, specplane;
    size_t qbuf;                      // SGP loop: the q planes are double-buffered, buffer s at in1 + s*qbuf (Ctrl::qsel)
    const cx<T> *tw;                  // exp(-2 pi i k / (nx/2)), k < nx/2
    const cx<T> *twh;                 // exp(-2 pi i k / nx),     k <= nx/2
    const T *alphaR;                  // boundary problems: alpha on R, 0 outside R (Eq.19-20)
    double *part, *part2;
    double bconst[kMaxP];
    int cy, cxs;                      // PSF centre (RFS_PSF)
    int check_status;                 // 1: return immediately when ct->status != 0
    unsigned int *btsync;             // K6: counters of the Armijo backtracking to re-arm (aux.cuh)
    const void *btinfo;               // K1 in the SGP loop: BtInfo<T> block in device memory (aux.cuh: Armijo backtracking)
    int count_fft;                    // inverse row kernels of the loops: two-dimensional transforms completed by this launch and the column
                                      // pass before it (p + 1), added to Ctrl::nfft by one thread
    size_t slab, tr_slab;             // batched plans: bytes between the per-problem arrays / trace blocks of consecutive problems
};

// Batched plans (sgp_plan_create_batched; PAPER.md:385-389 solves four sub-domain problems): problem
// b = blockIdx.z.  Every per-problem array of problem b lies `slab` bytes behind the one of problem b - 1 (one slab per
// problem, identical layout); twiddle tables, transfer functions and boundary weights are shared.  The kernels work on
// this per-problem view of the pointers of the parameter block; slab = 0 and gridDim.z = 1 for an ordinary plan.
template <typename U> __device__ __forceinline__ U *bshift(U *p, size_t off)
{
    return p ? reinterpret_cast<U *>(reinterpret_cast<unsigned char *>(const_cast<typename std::remove_const<U>::type *>(p)) + off) : p;
}
template <typename T> struct RowPtrs {
    const T *in0, *in1, *in2, *in3;
    T *out0, *out1;
    cx<T> *spec;
    double *part, *part2;
    Ctrl *ct;
    Trace tr;
    unsigned int *btsync;
    const void *btinfo;
    bool act;                         // false in the padding lanes of a thread group (fft_core.cuh: group_threads): no global stores
};
template <typename T> __device__ __forceinline__ RowPtrs<T> row_ptrs(const RowParams<T> &P)
{
    const size_t off = (size_t)blockIdx.z * P.slab, toff = (size_t)blockIdx.z * P.tr_slab;
    RowPtrs<T> X;
    X.in0 = bshift(P.in0, off); X.in1 = bshift(P.in1, off); X.in2 = bshift(P.in2, off); X.in3 = bshift(P.in3, off);
    X.out0 = bshift(P.out0, off); X.out1 = bshift(P.out1, off); X.spec = bshift(P.spec, off);
    X.part = bshift(P.part, off); X.part2 = bshift(P.part2, off); X.ct = bshift(P.ct, off);
    X.btsync = bshift(P.btsync, off); X.btinfo = bshift(P.btinfo, off);
    X.tr.J = bshift(P.tr.J, toff); X.tr.alpha = bshift(P.tr.alpha, toff); X.tr.lambda = bshift(P.tr.lambda, toff);
    X.tr.rule = bshift(P.tr.rule, toff); X.tr.backtracks = bshift(P.tr.backtracks, toff);
    X.tr.force_alpha = bshift(P.tr.force_alpha, toff); X.tr.force_lambda = bshift(P.tr.force_lambda, toff);
    X.tr.err = bshift(P.tr.err, toff);
    X.act = true;
    return X;
}

template <typename T> struct ColParams {
    Geom G;
    Ctrl *ct;
    const cx<T> *in;                  // spectrum of image j at + j*specplane
    cx<T> *out;
    const cx<T> *khat;                // tiled transfer function of image j at + j*specplane (scaled by 1/(ny nx))
    const cx<T> *khatB;               // column-0 companion of image j at + j*ny
    size_t specplane;
    const cx<T> *tw;                  // exp(-2 pi i k / ny)
    cx<T> *pack;                      // ny entries of scratch for the packed column of tile 0
    int p;
    int ntiles;                       // (nx/2)/C
    int check_status;
    size_t slab;                      // batched plans: bytes between the per-problem arrays (in, out, pack, ct) of consecutive problems
    int pf_ahead;                     // > 0: CTA b asks L2 for the tiles of CTA b + pf_ahead (the next wave) once its own have landed
};

// ---------------------------------------------------------------- elementwise pieces
// One summand of Eq.2: g ln(g/y) + y - g with y = A f + b, evaluated without
// cancellation (A17): g = 0 gives y; y <= 0 drops the log term.
__device__ __forceinline__ double kl_term(double g, double y)
{
    if (!(g > 0.0)) return y;
    if (!(y > 0.0)) return y - g;
    double t = (y - g) / g;
    return g * (t - log1p(t));
}
__device__ __forceinline__ float fast_rcp_f(float y) { float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(y)); return r; }
// float version: with u = (y-g)/(y+g), ln(y/g) = 2 atanh(u), hence
//   g ln(g/y) + y - g = u [ (y-g) - 2 g u^2 (1/3 + u^2/5 + u^4/7 + ...) ]      (u^2 < 0.09: 9 terms, < 1 ulp)
// and the plain form (y-g) - g log1p((y-g)/g) otherwise (no cancellation there).
__device__ __forceinline__ float kl_term(float g, float y)
{
    if (!(g > 0.f)) return y;
    if (!(y > 0.f)) return y - g;
    const float dy = y - g;
    const float u = __fdividef(dy, y + g);
    const float w = u * u;
    if (w < 0.09f) {
        float S = fmaf(w, 1.f / 19.f, 1.f / 17.f);
        S = fmaf(w, S, 1.f / 15.f);
        S = fmaf(w, S, 1.f / 13.f);
        S = fmaf(w, S, 1.f / 11.f);
        S = fmaf(w, S, 1.f / 9.f);
        S = fmaf(w, S, 1.f / 7.f);
        S = fmaf(w, S, 1.f / 5.f);
        S = fmaf(w, S, 1.f / 3.f);
        return u * (dy - 2.f * g * w * S);
    }
    return dy - g * log1pf(dy / g);
}
// Fast float path, valid for g > 0, y > 0, u^2 < 0.36 (y/g between 1/4 and 4: all but ~1e-4 of the pixels of a
// Poisson image with a background of 10 counts or more): S(w) = (atanh(u)/u - 1)/w by a degree-7 polynomial fitted
// on [0, 0.36] (max. relative error 9e-8 in float Horner arithmetic), u by the hardware reciprocal (1 ulp).
__device__ __forceinline__ float kl_series(float g, float y, bool &ok)
{
    const float dy = y - g;
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(y + g));
    const float u = dy * r;
    const float w = u * u;
    ok = (g > 0.f) && (y > 0.f) && (w < 0.36f);
    float S = fmaf(w, 2.629362187e-01f, -8.657711682e-02f);
    S = fmaf(w, S, 1.295689961e-01f);
    S = fmaf(w, S, 8.138694077e-02f);
    S = fmaf(w, S, 1.120216455e-01f);
    S = fmaf(w, S, 1.428151035e-01f);
    S = fmaf(w, S, 2.000007303e-01f);
    S = fmaf(w, S, 3.333333313e-01f);
    return u * fmaf(-2.f * g * w, S, dy);
}
// Pixels outside the range of kl_series: for y/g < 1/4 or > 4 the two terms of (y - g) - g ln(y/g) do not cancel (the
// result is >= 0.16 g), so the logarithm may come from the hardware lg2 (relative error 2^-22 outside (1/2, 2)): 4
// instructions instead of the ~60 of a division and log1pf -- a rejected Armijo trial, where most pixels overshoot,
// ran 3-4 times longer than an accepted one.  g = 0 gives y; y <= 0 drops the log term (A17).
__device__ __forceinline__ float kl_far(float g, float y)
{
    if (!(g > 0.f)) return y;
    if (!(y > 0.f)) return y - g;
    float rg, lr;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(rg) : "f"(g));
    asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(lr) : "f"(y * rg));
    const float w = (y - g) * fast_rcp_f(y + g);
    if (w * w < 0.36f) return kl_term(g, y);          // denormal / overflow corner cases of the fast test: the exact form
    return fmaf(-0.69314718055994530942f * g, lr, y - g);
}
// sum of kl_term over the pixels of a quad selected by s[]: straight-line code for the common case (so that the
// compiler interleaves the four dependency chains), the far-range form only where a pixel needs it
__device__ __forceinline__ float kl_quad(const float (&g)[4], const float (&y)[4], const bool (&s)[4])
{
    float k[4]; bool ok[4];
#pragma unroll
    for (int c = 0; c < 4; ++c) k[c] = kl_series(g[c], y[c], ok[c]);
    if (!((ok[0] || !s[0]) && (ok[1] || !s[1]) && (ok[2] || !s[2]) && (ok[3] || !s[3]))) {
#pragma unroll
        for (int c = 0; c < 4; ++c) if (s[c] && !ok[c]) k[c] = kl_far(g[c], y[c]);
    }
    return ((s[0] ? k[0] : 0.f) + (s[1] ? k[1] : 0.f)) + ((s[2] ? k[2] : 0.f) + (s[3] ? k[3] : 0.f));
}
__device__ __forceinline__ double kl_quad(const double (&g)[4], const double (&y)[4], const bool (&s)[4])
{
    double r = 0.0;
#pragma unroll
    for (int c = 0; c < 4; ++c) if (s[c]) r += kl_term(g[c], y[c]);
    return r;
}

// reciprocal: hardware approximation (1 ulp, one MUFU instruction) in float, exact in double
__device__ __forceinline__ float fast_rcp(float y) { float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(y)); return r; }
__device__ __forceinline__ double fast_rcp(double y) { return 1.0 / y; }
// ratio g/(Af+b) of Eq.1/11; 0 where the denominator is <= 0 (A17).  float: g * rcp(y), 1.5 ulp, 2 instructions
// instead of the ~10 of an IEEE division (64 of them per thread and row)
__device__ __forceinline__ float ratio_term(float g, float y) { return (y > 0.f) ? g * fast_rcp(y) : 0.f; }
__device__ __forceinline__ double ratio_term(double g, double y) { return (y > 0.0) ? g / y : 0.0; }
template <typename T> __device__ __forceinline__ T clipT(T f, T L1, T L2) { return fmin(L2, fmax(L1, f)); }

template <typename T> __device__ __forceinline__ cx<T> ld2(const T *p) { return *reinterpret_cast<const cx<T> *>(p); }
template <typename T> __device__ __forceinline__ void st2(T *p, cx<T> v) { *reinterpret_cast<cx<T> *>(p) = v; }
template <typename T> __device__ __forceinline__ void st2_if(bool act, T *p, cx<T> v) { if (act) *reinterpret_cast<cx<T> *>(p) = v; }

// W = M_R / alpha (Eq.21/23) for the two pixels of a pair; unmasked: 1/p.  r0, r1 = pixel in R.
template <typename T>
__device__ __forceinline__ void weights(const Geom &G, const T *alphaR, size_t idx, T Wc, cx<T> &a2, cx<T> &w2, bool &r0, bool &r1)
{
    r0 = true; r1 = true;
    w2 = mk<T>(Wc, Wc);
    if (G.masked) {
        a2 = ld2<T>(alphaR + idx);
        r0 = a2.x > (T)0; r1 = a2.y > (T)0;
        w2.x = r0 ? (T)1 / a2.x : (T)0; w2.y = r1 ? (T)1 / a2.y : (T)0;
    }
}

// Programmatic dependent launch (sm_90+): pdl_trigger lets the next kernel of the stream be scheduled once every CTA
// of this one has started, so that its CTAs fill the SMs as ours drain; pdl_wait blocks until the previous kernel
// has completed and its writes are visible.  Both are no-ops in a launch without the attribute.
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

__device__ __forceinline__ void prefetch_l2(const void *p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }
__device__ __forceinline__ void prefetch_l1(const void *p) { asm volatile("prefetch.global.L1 [%0];" ::"l"(p)); }
// The twiddle tables of a kernel on their way into the L1 at its start, one 128-byte line per thread.  The L1 is empty at
// every launch, and a CTA of the column kernel lives for one or two tiles only: 28 % of its twiddle sectors missed (ncu,
// 2048^2), each miss a trip to L2 in the middle of a pass.  Issued while the tile is still in flight, the trips overlap.
#ifndef SGP_TW_PREFETCH
#define SGP_TW_PREFETCH 1
#endif
template <typename C> __device__ __forceinline__ void prefetch_table_l1(const C *table, int entries, int tid, int nthr)
{
#if SGP_TW_PREFETCH
    const char *b = reinterpret_cast<const char *>(table);
    const int nlines = (entries * (int)sizeof(C) + 127) / 128;
    for (int l = tid; l < nlines; l += nthr) prefetch_l1(b + 128 * l);
#endif
}
// start one row of a plane (len reals) on its way to L2; called by the TF threads of the row
template <typename T> __device__ __forceinline__ void prefetch_row_l2(const T *row, int len, int t, int TF)
{
    constexpr int per_line = 128 / (int)sizeof(T);
    for (int i = t * per_line; i < len; i += TF * per_line) prefetch_l2(row + i);
}

// division that may be 2 ulp off in float (no slow path, no branch); exact in double
__device__ __forceinline__ float fast_div(float a, float b) { return a * fast_rcp(b); }
__device__ __forceinline__ double fast_div(double a, double b) { return a / b; }

// four consecutive pixels of a row
template <typename T> struct alignas(16) Quad { T a[4]; };
template <typename T> __device__ __forceinline__ Quad<T> ldq(const T *p) { return *reinterpret_cast<const Quad<T> *>(p); }
template <typename T> __device__ __forceinline__ void stq(T *p, const Quad<T> &v) { *reinterpret_cast<Quad<T> *>(p) = v; }
template <typename T> __device__ __forceinline__ void stq_if(bool act, T *p, const Quad<T> &v) { if (act) *reinterpret_cast<Quad<T> *>(p) = v; }

// address of spectrum entry (ky, kx) in the column-tile-major layout
__device__ __forceinline__ size_t spec_index(const Geom &G, int ky, int kx)
{
    return ((size_t)(kx >> G.lc) * (size_t)G.ny + (size_t)ky) * (size_t)G.C + (size_t)(kx & (G.C - 1));
}

}  // namespace sgpk
