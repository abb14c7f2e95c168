// small_params.h -- parameter block and look-up of the one-cluster-per-problem SGP kernel of the small grids (small.cuh);
// what the host side (plan_impl.inl) needs of it
#pragma once
#include "ew.cuh"

namespace sgpk {

template <typename T> struct SmallParams {
    Geom G; DevOpts o; Trace tr; Ctrl *ct;
    T *f, *grad, *d, *q;              // planes of problem 0 (q: both buffers, Ctrl::qsel says which is current)
    const T *g;
    const T *alphaR;                  // boundary problems: alpha on R, 0 outside (shared by the problems of a batch)
    size_t qbuf;
    const cx<T> *khat, *khatB;        // transfer function (tile-major, scaled by 1/(ny nx)) and its packed-column companion
    const cx<T> *tw_r, *tw_h, *tw_c;  // pass tables of the row / column FFTs, exp(-2 pi i k/nx)
    double bconst;                    // background of problem 0 (batched plans: Ctrl::bconst[0] of each problem)
    int iters;                        // iterations of this launch at most
    size_t slab, tr_slab;             // batched plans: bytes between the arrays / trace blocks of consecutive problems
    unsigned long long *dbg;          // developer builds (-DSGP_SMALL_TIMING): %globaltimer at the phase boundaries of one iteration
};

template <typename T> using small_kernel_t = void (*)(const SmallParams<T>);
// kernel for this geometry (nullptr: none), its cluster size, threads per CTA, dynamic shared memory and the elements per thread of
// its row / column FFT plans (fft_core.cuh: plan_radix), whose pass tables the host supplies
// two: the form compiled for two resident CTAs per SM (larger batches)
template <typename T> small_kernel_t<T> get_small(int ny, int nx, bool masked, bool rl, bool two, int *nc, int *threads, size_t *smem, int *er, int *ec);


}  // namespace sgpk
