// col.cuh -- column pass of FFT2 fused with the transfer-function product.
// A tile of C adjacent columns of the half spectrum is handled by one CTA: forward column FFTs, pointwise product
// with the transfer function(s) (conjugated and summed over the images for A^T), inverse column FFTs -- the
// spectrum never leaves the registers between the three steps.
//
// The kernel is PERSISTENT: grid = min(tiles, SMs), CTA b works on tiles b, b + grid, ...; the spectrum and the
// transfer-function tile of the next unit of work are copied global -> shared by the TMA engine (cp.async.bulk)
// while the current one is transformed, so the only exposed load is the first.  block = C * (L/E) threads (thread = (t, c), c
// fastest: global accesses are contiguous), dynamic smem = C * padded(L) complex (exchange buffer of the FFT
// passes) + 2 tiles (landing zones of the asynchronous copies).
//   CM_FWD / CM_INV: out = forward / unnormalised inverse column FFT of in (set-up of the transfer functions, rfft2 helpers)
//   CM_CONJSUM: out = IFFTcol( sum_j conj(K^_j) o FFTcol(in_j) )         (a2: sum_j A_j^T r_j in Fourier space, Eq.17)
//   CM_MULT   : out_j = IFFTcol( K^_j o FFTcol(in) ), j < p              (a8: A_j d, Eq.16)
// Column 0 of tile 0 carries the packed pair (kx = 0, kx = nx/2): with C~[ky] = conj(C[-ky]) the product is
//   C'[ky] = A[ky] C[ky] + B[ky] C~[ky],  A = (K0 + KM)/2 (stored in column 0 of khat), B = (K0 - KM)/2 (khatB).
// The partner values C[-ky] of that one column go through a small global scratch line (P.pack, L entries).
#pragma once
#include "ew.cuh"

namespace sgpk {

enum ColMode { CM_FWD = 0, CM_CONJSUM = 1, CM_MULT = 2, CM_INV = 3 };

// option: pass twiddles of the float column transforms from a few table entries and one product each (fft_core.cuh: TWP).
// K2 / K5 43.3 / 40.2 -> 39.5 / 36.8 us at 3 x 2048^2 (the image loop repeats the passes p times per tile); OFF: it changes the
// rounding of every transform, and that was enough to move the long free-running fp32 parity runs
#ifndef SGP_COL_TWP
#define SGP_COL_TWP 0
#endif
#ifndef SGP_TWP_F64
#define SGP_TWP_F64 0      // experiment: the same in the double kernels
#endif
template <typename T> constexpr bool kColTwp = SGP_COL_TWP && (sizeof(T) == 4 || SGP_TWP_F64);
// experiment: the tiles of the NEXT wave of CTAs requested into L2 by the CTAs of this one (ColParams::pf_ahead), so that DRAM
// works while the SMs transform instead of idling until the next wave asks for its tiles all at once.  Measured: K2 / K5
// 43.3 / 40.2 -> 42.2 / 39.0 us at 3 x 2048^2, 22.9 / 20.9 -> 23.0 / 21.3 us at 2048^2 (RL 13 360 -> 13 260 it/s): off
#ifndef SGP_COL_PF2
#define SGP_COL_PF2 0
#endif
__device__ __forceinline__ void bulk_prefetch_l2(const void *gmem, unsigned int bytes)
{
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(gmem), "r"(bytes) : "memory");
}

// Bulk asynchronous copy global -> shared by the TMA engine (cp.async.bulk, SASS UBLKCP): ONE instruction of one
// thread moves a whole tile (contiguous in the tile-major layout); completion is signalled on an mbarrier.
__device__ __forceinline__ unsigned int smem_u32(const void *p) { return (unsigned int)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long *bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void bulk_load(void *smem_dst, const void *gmem_src, unsigned int bytes, unsigned long long *bar)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(smem_dst)), "l"(gmem_src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long *bar, unsigned int phase)
{
    unsigned int ok;
    do {
        asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
                     : "=r"(ok) : "r"(smem_u32(bar)), "r"(phase) : "memory");
    } while (!ok);
}

// per-CTA view of the work: tile it of this CTA starts at tile_of(it) in a spectrum plane
template <typename T, int L, int E, bool BATCH> struct ColCtx {
    using C = cx<T>;
    int tid, nthr, t, c, Cc;
    size_t tile_len;
    size_t zoff;                      // batched plans: offset (in complex numbers) of problem blockIdx.z's spectra behind problem 0's
    C *smc, *bufA, *bufB;
    // tile `it` of this CTA in the shared transfer function / in this problem's spectra
    __device__ __forceinline__ size_t ktile_of(int it) const { return (size_t)((int)blockIdx.x + it * (int)gridDim.x) * tile_len; }
    __device__ __forceinline__ size_t tile_of(int it) const { if constexpr (BATCH) return zoff + ktile_of(it); else return ktile_of(it); }
};

// product with the packed-column companion B (see the header): r[e] (+)= conj?(B) C~
template <typename T, int L, int E, bool CONJ>
__device__ __forceinline__ void packed_fix(cx<T> (&r)[E], volatile cx<T> *pack, const cx<T> *khatB, int t)
{
    using C = cx<T>;
    constexpr int TF = L / E;
#pragma unroll
    for (int e = 0; e < E; ++e) {
        const int ky = t + TF * e, kyn = ky == 0 ? 0 : L - ky;
        C ct; ct.x = pack[kyn].x; ct.y = -pack[kyn].y;
        r[e] = cadd(r[e], CONJ ? cmulc(ct, khatB[ky]) : cmul(ct, khatB[ky]));
    }
}

// tile width the host chooses by default (api.cu: choose_tiles) for this element type and length: with it known at
// compile time the shared-memory addresses of the exchanges are immediates (no spills, fewer integer instructions)
template <typename T> __host__ __device__ constexpr int col_default_C(int L)
{
    const int E = fft_E_col<T>(L), TF = L / E, col_max = E == 32 ? 256 : 512;
    int C = 1;
    while (2 * C <= (col_max / TF > 1 ? col_max / TF : 1) && 2 * C <= 32) C *= 2;
    while (C > 1 && (size_t)C * fft_padded_len(L, E) * sizeof(cx<T>) > 72 * 1024) C /= 2;
    while (C > 8 && (L / 2) / C < 32) C /= 2;          // small grids (api.cu: choose_tiles), assuming nx = ny
    return C;
}

// BATCH: a batched plan (blockIdx.z = problem, ew.cuh).  A template parameter because the product kernels sit exactly at
// their register limit: the two registers of a run-time batch offset made them spill (K2 at 3 x 2048^2: 39 -> 52 us).
template <typename T, int L, int MODE, bool MULTI, int CT, bool BATCH>
__device__ __forceinline__ void col_body(const ColParams<T> &P)
{
    using C = cx<T>;
    constexpr int E = fft_E_col<T>(L);
    constexpr int TF = L / E;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C *sm = reinterpret_cast<C *>(smem_raw);
    pdl_trigger();

    ColCtx<T, L, E, BATCH> X;
    X.Cc = CT > 0 ? CT : P.G.C; X.tid = threadIdx.x; X.nthr = CT > 0 ? CT * TF : (int)blockDim.x;
    X.t = X.tid / X.Cc; X.c = X.tid - X.t * X.Cc;
    X.tile_len = (size_t)L * X.Cc;
    if constexpr (BATCH) X.zoff = (size_t)blockIdx.z * (P.slab / sizeof(C));      // batched plans (ew.cuh)
    X.smc = sm + X.c;
    X.bufA = sm + (size_t)X.Cc * fft_padded_len(L, E);     // landing zone of the spectrum tile
    X.bufB = X.bufA + X.tile_len;                          // landing zone of the transfer-function tile
    const int tid = X.tid, nthr = X.nthr, t = X.t, Cc = X.Cc;
    volatile C *pack = (BATCH ? bshift(P.pack, (size_t)blockIdx.z * P.slab) : P.pack);
    const SyncBlock sync;
    const int ntiles = P.ntiles;
    C v[E];

    if constexpr (MODE == CM_FWD || MODE == CM_INV) {
        pdl_wait();
        for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
            const size_t tbase = (BATCH ? X.zoff : 0) + (size_t)tile * X.tile_len + tid;
#pragma unroll
            for (int e = 0; e < E; ++e) v[e] = P.in[tbase + (size_t)e * nthr];
            fft_block<T, L, E, (MODE == CM_FWD ? -1 : +1)>(v, X.smc, Cc, t, P.tw, sync);
#pragma unroll
            for (int e = 0; e < E; ++e) P.out[tbase + (size_t)e * nthr] = v[e];
        }
        return;
    }
    const int p = MULTI ? P.p : 1;
    const int my_tiles = ((int)blockIdx.x < ntiles) ? (ntiles - 1 - (int)blockIdx.x) / (int)gridDim.x + 1 : 0;
    if (my_tiles == 0) return;
    // landing zones: bufA <- spectrum tile, bufB <- transfer-function tile, one mbarrier each.  Thread 0 issues the
    // copies; a zone is re-filled only after a CTA barrier that follows the last read of it.
    __shared__ unsigned long long bars[2];
    const unsigned int tile_bytes = (unsigned int)(X.tile_len * sizeof(C));
    unsigned int phA = 0, phB = 0;
    if (tid == 0) {
        mbar_init(&bars[0], 1); mbar_init(&bars[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        // the transfer function does not depend on the previous kernel: it is on its way before we wait for that
        bulk_load(X.bufB, P.khat + X.ktile_of(0), tile_bytes, &bars[1]);
    }
    pdl_wait();
    // (The transforms are counted by the inverse row kernel that follows every column pass, and this test is kept as simple
    // as it is: anything more in this kernel keeps the compiler from hoisting the first twiddle loads above the wait for
    // the tile -- K2 / K5 45 instead of 39 us at 3 x 2048^2.  The refresh round of reading A21 passes a shadow control block
    // whose status says "not this iteration".)
    const int stop = P.check_status ? (BATCH ? bshift(P.ct, (size_t)blockIdx.z * P.slab) : P.ct)->status : 0;
    if (tid == 0 && stop == 0) bulk_load(X.bufA, P.in + X.tile_of(0), tile_bytes, &bars[0]);
    __syncthreads();                                            // barrier initialisation visible to all
    if (stop != 0) { mbar_wait(&bars[1], 0); return; }

    if constexpr (MODE == CM_CONJSUM) {
        // unit of work u = it*p + j: spectrum and transfer function of image j on this CTA's it-th tile
        const int units = my_tiles * p;
        C acc[MULTI ? E : 1];
        for (int it = 0; it < my_tiles; ++it) {
            const bool packed = (blockIdx.x == 0 && it == 0);      // tile 0 holds the packed column
            const bool pk = packed && X.c == 0;
            for (int j = 0; j < p; ++j) {
                const int u1 = it * p + j + 1, it1 = u1 / p, j1 = u1 - it1 * p;
                mbar_wait(&bars[0], phA); phA ^= 1;                 // spectrum of this unit has landed
                if constexpr (SGP_COL_PF2 != 0) {
                    if (tid == 0 && it == 0 && j == 0 && P.pf_ahead > 0 && (int)blockIdx.x + P.pf_ahead < ntiles) {
                        const size_t t2 = (size_t)P.pf_ahead * X.tile_len;
                        for (int jj = 0; jj < p; ++jj) {
                            bulk_prefetch_l2(P.in + (size_t)jj * P.specplane + X.tile_of(0) + t2, tile_bytes);
                            bulk_prefetch_l2(P.khat + (size_t)jj * P.specplane + X.ktile_of(0) + t2, tile_bytes);
                        }
                    }
                }
#pragma unroll
                for (int e = 0; e < E; ++e) v[e] = X.bufA[tid + e * nthr];
                if (u1 < units) {
                    __syncthreads();
                    if (tid == 0) bulk_load(X.bufA, P.in + (size_t)j1 * P.specplane + X.tile_of(it1), tile_bytes, &bars[0]);
                }
                fft_block<T, L, E, -1, false, kColTwp<T>>(v, X.smc, Cc, t, P.tw, sync);
                if (packed) {
                    if (pk) {
#pragma unroll
                        for (int e = 0; e < E; ++e) { pack[t + TF * e].x = v[e].x; pack[t + TF * e].y = v[e].y; }
                    }
                    __syncthreads();
                }
                mbar_wait(&bars[1], phB); phB ^= 1;                 // transfer function of this unit has landed
#pragma unroll
                for (int e = 0; e < E; ++e) v[e] = cmulc(v[e], X.bufB[tid + e * nthr]);
                if (u1 < units) {
                    __syncthreads();
                    if (tid == 0) bulk_load(X.bufB, P.khat + (size_t)j1 * P.specplane + X.ktile_of(it1), tile_bytes, &bars[1]);
                }
                if (pk) packed_fix<T, L, E, true>(v, pack, P.khatB + (size_t)j * L, t);
                if constexpr (MULTI) {
#pragma unroll
                    for (int e = 0; e < E; ++e) acc[e] = (j == 0) ? v[e] : cadd(acc[e], v[e]);
                    if (packed) __syncthreads();                    // pack[] is rewritten for the next image
                }
            }
            if constexpr (MULTI) {
#pragma unroll
                for (int e = 0; e < E; ++e) v[e] = acc[e];
            }
            fft_block<T, L, E, +1, false, kColTwp<T>>(v, X.smc, Cc, t, P.tw, sync);
            C *dst = P.out + X.tile_of(it) + tid;
#pragma unroll
            for (int e = 0; e < E; ++e) dst[(size_t)e * nthr] = v[e];
        }
    } else {   // CM_MULT
        for (int it = 0; it < my_tiles; ++it) {
            const bool packed = (blockIdx.x == 0 && it == 0);
            const bool pk = packed && X.c == 0;
            mbar_wait(&bars[0], phA); phA ^= 1;                     // spectrum of tile it has landed
            if constexpr (SGP_COL_PF2 != 0) {
                if (tid == 0 && it == 0 && P.pf_ahead > 0 && (int)blockIdx.x + P.pf_ahead < ntiles) {
                    const size_t t2 = (size_t)P.pf_ahead * X.tile_len;
                    bulk_prefetch_l2(P.in + X.tile_of(0) + t2, tile_bytes);
                    for (int jj = 0; jj < p; ++jj) bulk_prefetch_l2(P.khat + (size_t)jj * P.specplane + X.ktile_of(0) + t2, tile_bytes);
                }
            }
#pragma unroll
            for (int e = 0; e < E; ++e) v[e] = X.bufA[tid + e * nthr];
            if (it + 1 < my_tiles) {
                __syncthreads();
                if (tid == 0) bulk_load(X.bufA, P.in + X.tile_of(it + 1), tile_bytes, &bars[0]);
            }
            fft_block<T, L, E, -1, false, kColTwp<T>>(v, X.smc, Cc, t, P.tw, sync);
            if (packed) {
                if (pk) {
#pragma unroll
                    for (int e = 0; e < E; ++e) { pack[t + TF * e].x = v[e].x; pack[t + TF * e].y = v[e].y; }
                }
                __syncthreads();
            }
            for (int j = 0; j < p; ++j) {
                C w[E];
                mbar_wait(&bars[1], phB); phB ^= 1;                 // transfer function (it, j) has landed
#pragma unroll
                for (int e = 0; e < E; ++e) w[e] = cmul(v[e], X.bufB[tid + e * nthr]);
                if (j + 1 < p || it + 1 < my_tiles) {
                    __syncthreads();
                    if (tid == 0) {
                        if (j + 1 < p) bulk_load(X.bufB, P.khat + (size_t)(j + 1) * P.specplane + X.ktile_of(it), tile_bytes, &bars[1]);
                        else           bulk_load(X.bufB, P.khat + X.ktile_of(it + 1), tile_bytes, &bars[1]);
                    }
                }
                if (pk) packed_fix<T, L, E, false>(w, pack, P.khatB + (size_t)j * L, t);
                fft_block<T, L, E, +1, false, kColTwp<T>>(w, X.smc, Cc, t, P.tw, sync);
                C *dst = P.out + (size_t)j * P.specplane + X.tile_of(it) + tid;
#pragma unroll
                for (int e = 0; e < E; ++e) dst[(size_t)e * nthr] = w[e];
            }
        }
    }
}

// CT = 0: tile width from P.G.C; CT > 0: compiled for that width (the host launches it only when G.C == CT)
template <typename T, int L, int MODE, bool MULTI, int CT = 0, bool BATCH = false>
__global__ void __launch_bounds__(fft_E_col<T>(L) == 32 ? 256 : 512, 1) col_kernel(const ColParams<T> P)
{
    col_body<T, L, MODE, MULTI, CT, BATCH>(P);
}

// ---------------------------------------------------------------------------------------------------------------
// Second form of the column pass for single-image problems (CM_CONJSUM / CM_MULT with p = 1), float:
// 32 elements per thread (passes 32 x 8 x 8 at L = 2048), 256 threads per CTA, and only ONE shared-memory buffer --
// the landing zone of the spectrum tile is the exchange buffer of the FFT passes, the transfer function comes
// straight from global memory (L2-resident: it is read twice per iteration) into the registers.  68 KB and 128
// registers per CTA, so TWO CTAs share an SM: the whole grid (256 tiles at 2048^2) is resident at once instead of
// 1.73 waves of one 200 KB CTA per SM, and one CTA's loads and stores overlap the other's butterflies.
template <typename T, int L, int MODE, bool BATCH = false>
__global__ void __launch_bounds__(256, 2) col2_kernel(const ColParams<T> P)
{
    using C = cx<T>;
    static_assert(MODE == CM_CONJSUM || MODE == CM_MULT, "col2_kernel: product modes only");
    constexpr int E = 32;
    constexpr int TF = L / E;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    C *sm = reinterpret_cast<C *>(smem_raw);
    __shared__ unsigned long long bar;
    constexpr int Cc = 256 / TF, nthr = 256;                    // tile width fixed by the block size (the host checks G.C)
    const int tid = threadIdx.x;
    const int t = tid / Cc, c = tid - t * Cc;
    constexpr size_t tile_len = (size_t)L * Cc;
    const size_t kbase = (size_t)blockIdx.x * tile_len;                              // in the (shared) transfer function
    const size_t tbase = kbase + (BATCH ? (size_t)blockIdx.z * (P.slab / sizeof(C)) : 0);          // in this problem's spectra (batched plans)
    const unsigned int tile_bytes = (unsigned int)(tile_len * sizeof(C));
    {
        Ctrl *ctz = BATCH ? bshift(P.ct, (size_t)blockIdx.z * P.slab) : P.ct;
        const int stop = P.check_status ? ctz->status : 0;
        if (stop != 0) return;
    }
    if (tid == 0) {
        mbar_init(&bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        bulk_load(sm, P.in + tbase, tile_bytes, &bar);
        // the transfer-function tile is wanted after the forward transform: start it on its way to L2 now (in the SGP
        // loop the planes touched since its last use have pushed it out to HBM)
        asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(P.khat + kbase), "r"(tile_bytes) : "memory");
    }
    __syncthreads();                                            // barrier initialisation visible to all
    const SyncBlock sync;
    const bool packed = blockIdx.x == 0;                        // tile 0 holds the packed column (kx = 0 and nx/2)
    const bool pk = packed && c == 0;
    volatile C *pack = (BATCH ? bshift(P.pack, (size_t)blockIdx.z * P.slab) : P.pack);
    C v[E];
    mbar_wait(&bar, 0);
#pragma unroll
    for (int e = 0; e < E; ++e) v[e] = sm[tid + e * nthr];
    fft_block<T, L, E, -1>(v, sm + c, Cc, t, P.tw, sync);       // its first exchange starts with a barrier: the tile has been read
    if (packed) {
        if (pk) {
#pragma unroll
            for (int e = 0; e < E; ++e) { pack[t + TF * e].x = v[e].x; pack[t + TF * e].y = v[e].y; }
        }
        __syncthreads();
    }
    const C *kh = P.khat + kbase + tid;
#pragma unroll
    for (int e0 = 0; e0 < E; e0 += 8) {
        C k[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) k[u] = __ldg(&kh[(size_t)(e0 + u) * nthr]);
#pragma unroll
        for (int u = 0; u < 8; ++u) v[e0 + u] = (MODE == CM_CONJSUM) ? cmulc(v[e0 + u], k[u]) : cmul(v[e0 + u], k[u]);
    }
    if (pk) packed_fix<T, L, E, MODE == CM_CONJSUM>(v, pack, P.khatB, t);
    fft_block<T, L, E, +1>(v, sm + c, Cc, t, P.tw, sync);
    C *dst = P.out + tbase + tid;
#pragma unroll
    for (int e = 0; e < E; ++e) dst[(size_t)e * nthr] = v[e];
}

}  // namespace sgpk
