// col.cuh -- column pass of FFT2 fused with the transfer-function product.
// One CTA owns a tile of C adjacent columns of the half spectrum: forward column FFTs, pointwise product with
// the transfer function(s) (conjugated and summed over the images for A^T), inverse column FFTs -- the spectrum
// never leaves the registers between the three steps.
//
// grid = (nx/2)/C tiles, block = C * (L/E) threads (thread = (t, c), c fastest, so global accesses are
// contiguous), dynamic smem = C * padded(L) complex.
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

__device__ __forceinline__ void prefetch_l2(const void *p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }

template <typename T, int L, int MODE, bool MULTI>
__global__ void __launch_bounds__(fft_E_col<T>(L) == 32 ? 256 : 512, ((fft_E_col<T>(L) == 32 && !MULTI) || (fft_E_col<T>(L) == 8 && sizeof(T) == 4)) ? 2 : 1) col_kernel(const ColParams<T> P)
{
    using C = cx<T>;
    constexpr int E = fft_E_col<T>(L);
    constexpr int TF = L / E;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C *sm = reinterpret_cast<C *>(smem_raw);
    if (P.check_status && P.ct->status != 0) return;

    const int Cc = P.G.C;
    const int tid = threadIdx.x, nthr = blockDim.x;
    const int t = tid / Cc, c = tid - t * Cc;
    const size_t tbase = (size_t)blockIdx.x * ((size_t)L * Cc) + tid;
    C *smc = sm + c;
    const bool packed = (blockIdx.x == 0);      // tile 0 holds the packed column
    const bool pk = packed && c == 0;
    volatile C *pack = P.pack;
    const SyncBlock sync;
    C v[E];

    if constexpr (MODE == CM_FWD || MODE == CM_INV) {
#pragma unroll
        for (int e = 0; e < E; ++e) v[e] = P.in[tbase + (size_t)e * nthr];
        fft_block<T, L, E, (MODE == CM_FWD ? -1 : +1)>(v, smc, Cc, t, P.tw, sync);
#pragma unroll
        for (int e = 0; e < E; ++e) P.out[tbase + (size_t)e * nthr] = v[e];
    } else if constexpr (MODE == CM_CONJSUM) {
        C acc[MULTI ? E : 1];
        const int p = MULTI ? P.p : 1;
        for (int j = 0; j < p; ++j) {
            const C *src = P.in + (size_t)j * P.specplane;
            const C *kh = P.khat + (size_t)j * P.specplane;
#pragma unroll
            for (int e = 0; e < E; ++e) v[e] = src[tbase + (size_t)e * nthr];
            // the transfer function is needed only after the forward transform: start it on its way to L2 now
            for (int e = (tid & 15); e < E; e += 16) prefetch_l2(kh + tbase - (tid & 15) + (size_t)e * nthr);
            fft_block<T, L, E, -1>(v, smc, Cc, t, P.tw, sync);
            if (packed) {
                if (pk) {
#pragma unroll
                    for (int e = 0; e < E; ++e) { pack[t + TF * e].x = v[e].x; pack[t + TF * e].y = v[e].y; }
                }
                __syncthreads();
            }
#pragma unroll
            for (int e = 0; e < E; ++e) {
                const C k = kh[tbase + (size_t)e * nthr];
                const C r = cmulc(v[e], k);
                if constexpr (MULTI) { if (j == 0) acc[e] = r; else acc[e] = cadd(acc[e], r); }
                else v[e] = r;
            }
            if (pk) {
#pragma unroll
                for (int e = 0; e < E; ++e) {
                    const int ky = t + TF * e, kyn = ky == 0 ? 0 : L - ky;
                    C ct; ct.x = pack[kyn].x; ct.y = -pack[kyn].y;
                    const C r = cmulc(ct, P.khatB[(size_t)j * L + ky]);
                    if constexpr (MULTI) acc[e] = cadd(acc[e], r); else v[e] = cadd(v[e], r);
                }
            }
            if (packed && MULTI) __syncthreads();      // pack[] is rewritten for the next image
        }
        if constexpr (MULTI) {
#pragma unroll
            for (int e = 0; e < E; ++e) v[e] = acc[e];
        }
        fft_block<T, L, E, +1>(v, smc, Cc, t, P.tw, sync);
#pragma unroll
        for (int e = 0; e < E; ++e) P.out[tbase + (size_t)e * nthr] = v[e];
    } else {   // CM_MULT
#pragma unroll
        for (int e = 0; e < E; ++e) v[e] = P.in[tbase + (size_t)e * nthr];
        for (int e = (tid & 15); e < E; e += 16) prefetch_l2(P.khat + tbase - (tid & 15) + (size_t)e * nthr);
        fft_block<T, L, E, -1>(v, smc, Cc, t, P.tw, sync);
        if (packed) {
            if (pk) {
#pragma unroll
                for (int e = 0; e < E; ++e) { pack[t + TF * e].x = v[e].x; pack[t + TF * e].y = v[e].y; }
            }
            __syncthreads();
        }
        const int p = MULTI ? P.p : 1;
        for (int j = 0; j < p; ++j) {
            const C *kh = P.khat + (size_t)j * P.specplane;
            C w[E];
#pragma unroll
            for (int e = 0; e < E; ++e) w[e] = cmul(v[e], kh[tbase + (size_t)e * nthr]);
            if (pk) {
#pragma unroll
                for (int e = 0; e < E; ++e) {
                    const int ky = t + TF * e, kyn = ky == 0 ? 0 : L - ky;
                    C ct; ct.x = pack[kyn].x; ct.y = -pack[kyn].y;
                    w[e] = cadd(w[e], cmul(ct, P.khatB[(size_t)j * L + ky]));
                }
            }
            fft_block<T, L, E, +1>(w, smc, Cc, t, P.tw, sync);
            C *dst = P.out + (size_t)j * P.specplane;
#pragma unroll
            for (int e = 0; e < E; ++e) dst[tbase + (size_t)e * nthr] = w[e];
        }
    }
}

}  // namespace sgpk
