// fft_core.cuh -- register-resident Stockham FFT building blocks for sm_100a.
//
// One complex FFT of length L is computed by TF = L/E threads; every thread keeps E complex values in
// registers.  Contract of fft_passes<>: on entry v[e] = x[t + TF*e], on exit v[e] = X[t + TF*e]
// (t = the thread's index inside its FFT), i.e. both sides are in natural order with the SAME
// thread/register mapping, so forward transform -> pointwise multiply -> inverse transform needs no
// data movement in between.  Between two passes the values are exchanged through shared memory
// (autosort Stockham indexing: out[(j/Ns)*Ns*R + j%Ns + s*Ns], in[j + r*L/R]).
//
// This is the FFT that evaluates the convolutions A f and A^T y "by means of FFT".
#pragma once
#include <cuda_runtime.h>

namespace sgpk {

template <typename T> struct cx_of;
template <> struct cx_of<float>  { using type = float2; };
template <> struct cx_of<double> { using type = double2; };
template <typename T> using cx = typename cx_of<T>::type;

template <typename T> __device__ __forceinline__ cx<T> mk(T a, T b) { cx<T> r; r.x = a; r.y = b; return r; }
template <typename C> __device__ __forceinline__ C cadd(C a, C b) { C r; r.x = a.x + b.x; r.y = a.y + b.y; return r; }
template <typename C> __device__ __forceinline__ C csub(C a, C b) { C r; r.x = a.x - b.x; r.y = a.y - b.y; return r; }
template <typename C> __device__ __forceinline__ C cmul(C a, C b) { C r; r.x = a.x * b.x - a.y * b.y; r.y = a.x * b.y + a.y * b.x; return r; }
// a * conj(b)
template <typename C> __device__ __forceinline__ C cmulc(C a, C b) { C r; r.x = a.x * b.x + a.y * b.y; r.y = a.y * b.x - a.x * b.y; return r; }
template <typename C> __device__ __forceinline__ C cconj(C a) { C r; r.x = a.x; r.y = -a.y; return r; }
// multiply by -i (forward, DIR = -1) or +i (inverse, DIR = +1)
template <int DIR, typename C> __device__ __forceinline__ C mul_dir_i(C a)
{
    C r;
    if (DIR < 0) { r.x = a.y; r.y = -a.x; } else { r.x = -a.y; r.y = a.x; }
    return r;
}
// multiply by cos - i sin (forward) or cos + i sin (inverse): the constant twiddle W_R^k with (c,s) = (cos, sin)(2 pi k / R)
template <int DIR, typename C, typename T> __device__ __forceinline__ C tw_const(C a, T c, T s)
{
    C r;
    if (DIR < 0) { r.x = a.x * c + a.y * s; r.y = a.y * c - a.x * s; }
    else         { r.x = a.x * c - a.y * s; r.y = a.y * c + a.x * s; }
    return r;
}

// ---------------------------------------------------------------- small DFTs, natural order in and out
template <int DIR, typename C> __device__ __forceinline__ void dft2(C &a0, C &a1)
{
    C t = a0; a0 = cadd(t, a1); a1 = csub(t, a1);
}
template <int DIR, typename C> __device__ __forceinline__ void dft4(C &a0, C &a1, C &a2, C &a3)
{
    C t0 = cadd(a0, a2), t1 = csub(a0, a2), t2 = cadd(a1, a3), t3 = mul_dir_i<DIR>(csub(a1, a3));
    a0 = cadd(t0, t2); a1 = cadd(t1, t3); a2 = csub(t0, t2); a3 = csub(t1, t3);
}
template <int DIR, typename T, typename C> __device__ __forceinline__ void dft5(C &a0, C &a1, C &a2, C &a3, C &a4)
{
    const T c1 = (T)0.30901699437494742410, c2 = (T)-0.80901699437494742410;   // cos(2pi/5), cos(4pi/5)
    const T s1 = (T)0.95105651629515357212, s2 = (T)0.58778525229247312917;    // sin(2pi/5), sin(4pi/5)
    C p1 = cadd(a1, a4), p2 = cadd(a2, a3), m1 = csub(a1, a4), m2 = csub(a2, a3);
    C r1, r2, q1, q2;
    r1.x = a0.x + c1 * p1.x + c2 * p2.x; r1.y = a0.y + c1 * p1.y + c2 * p2.y;
    r2.x = a0.x + c2 * p1.x + c1 * p2.x; r2.y = a0.y + c2 * p1.y + c1 * p2.y;
    q1.x = s1 * m1.x + s2 * m2.x; q1.y = s1 * m1.y + s2 * m2.y;
    q2.x = s2 * m1.x - s1 * m2.x; q2.y = s2 * m1.y - s1 * m2.y;
    a0.x = a0.x + p1.x + p2.x; a0.y = a0.y + p1.y + p2.y;
    C iq1 = mul_dir_i<DIR>(q1), iq2 = mul_dir_i<DIR>(q2);   // forward: -i q
    a1 = cadd(r1, iq1); a4 = csub(r1, iq1);
    a2 = cadd(r2, iq2); a3 = csub(r2, iq2);
}

// cos / sin of 2 pi k / 32 from the quarter-wave table (folded to immediates once the callers are unrolled)
__host__ __device__ constexpr double q32(int k)
{
    return k == 0 ? 1.0 : k == 1 ? 0.98078528040323043058 : k == 2 ? 0.92387953251128673848 : k == 3 ? 0.83146961230254523567
         : k == 4 ? 0.70710678118654752440 : k == 5 ? 0.55557023301960217765 : k == 6 ? 0.38268343236508978178
         : k == 7 ? 0.19509032201612824808 : 0.0;
}
__host__ __device__ constexpr double cos32(int k)
{
    k &= 31;
    return k <= 8 ? q32(k) : k <= 16 ? -q32(16 - k) : k <= 24 ? -q32(k - 16) : q32(32 - k);
}
__host__ __device__ constexpr double sin32(int k) { return cos32(k + 24); }
// cos / sin of 2 pi k / 64, 0 <= k <= 16 (the real<->complex step of a row whose threads hold 32 elements: row_fwd.cuh, SGP_ROW_TWC)
__host__ __device__ constexpr double cos64q(int k)
{
    return k == 0 ? 1.0 : k == 1 ? 0.99518472667219688624 : k == 2 ? 0.98078528040323044913 : k == 3 ? 0.95694033573220886494
         : k == 4 ? 0.92387953251128675613 : k == 5 ? 0.88192126434835502971 : k == 6 ? 0.83146961230254523708
         : k == 7 ? 0.77301045336273696081 : k == 8 ? 0.70710678118654752440 : k == 9 ? 0.63439328416364549822
         : k == 10 ? 0.55557023301960222474 : k == 11 ? 0.47139673682599764856 : k == 12 ? 0.38268343236508977173
         : k == 13 ? 0.29028467725446236764 : k == 14 ? 0.19509032201612826785 : k == 15 ? 0.09801714032956060199 : 0.0;
}
__host__ __device__ constexpr double sin64q(int k) { return cos64q(16 - k); }

// 8-point DFT on references, natural order in and out
template <int DIR, typename T, typename C>
__device__ __forceinline__ void dft8r(C &a0, C &a1, C &a2, C &a3, C &a4, C &a5, C &a6, C &a7)
{
    const T h = (T)0.70710678118654752440;
    dft4<DIR>(a0, a2, a4, a6);
    dft4<DIR>(a1, a3, a5, a7);
    a3 = tw_const<DIR>(a3, h, h);
    a5 = mul_dir_i<DIR>(a5);
    a7 = tw_const<DIR>(a7, -h, h);
    dft2<DIR>(a0, a1); dft2<DIR>(a2, a3); dft2<DIR>(a4, a5); dft2<DIR>(a6, a7);
    // position 2*s1 + s2 holds X[s1 + 4*s2]
    C o1 = a2, o2 = a4, o3 = a6, o4 = a1, o5 = a3, o6 = a5, o7 = a7;
    a1 = o1; a2 = o2; a3 = o3; a4 = o4; a5 = o5; a6 = o6; a7 = o7;
}

// In-register DFT of R points, a[r] -> a[s] (natural order).  Composite radices are Cooley-Tukey
// products R = R1*R2 with input index r = R2*a + b and output index s = s1 + R1*s2.
template <int R, int DIR, typename T, typename C> __device__ __forceinline__ void dft(C (&a)[R])
{
    const T h = (T)0.70710678118654752440;   // sqrt(1/2)
    if constexpr (R == 2) {
        dft2<DIR>(a[0], a[1]);
    } else if constexpr (R == 4) {
        dft4<DIR>(a[0], a[1], a[2], a[3]);
    } else if constexpr (R == 5) {
        dft5<DIR, T>(a[0], a[1], a[2], a[3], a[4]);
    } else if constexpr (R == 8) {
        // R1 = 4 (over a), R2 = 2 (b): r = 2a + b
        dft4<DIR>(a[0], a[2], a[4], a[6]);
        dft4<DIR>(a[1], a[3], a[5], a[7]);
        a[3] = tw_const<DIR>(a[3], h, h);            // W8^1  (s1 = 1, b = 1)
        a[5] = mul_dir_i<DIR>(a[5]);                 // W8^2
        a[7] = tw_const<DIR>(a[7], -h, h);           // W8^3
        dft2<DIR>(a[0], a[1]); dft2<DIR>(a[2], a[3]); dft2<DIR>(a[4], a[5]); dft2<DIR>(a[6], a[7]);
        // position 2*s1 + s2 holds X[s1 + 4*s2]
        C o1 = a[2], o2 = a[4], o3 = a[6], o4 = a[1], o5 = a[3], o6 = a[5], o7 = a[7];
        a[1] = o1; a[2] = o2; a[3] = o3; a[4] = o4; a[5] = o5; a[6] = o6; a[7] = o7;
    } else if constexpr (R == 16) {
        // R1 = 4, R2 = 4: r = 4a + b
        const T c1 = (T)0.92387953251128675613, s1 = (T)0.38268343236508977173;   // cos, sin (pi/8)
#pragma unroll
        for (int b = 0; b < 4; ++b) dft4<DIR>(a[b], a[4 + b], a[8 + b], a[12 + b]);
        // u[4*s1 + b] *= W16^(b*s1)
        a[5]  = tw_const<DIR>(a[5], c1, s1);         // k = 1
        a[6]  = tw_const<DIR>(a[6], h, h);           // k = 2
        a[7]  = tw_const<DIR>(a[7], s1, c1);         // k = 3
        a[9]  = tw_const<DIR>(a[9], h, h);           // k = 2
        a[10] = mul_dir_i<DIR>(a[10]);               // k = 4
        a[11] = tw_const<DIR>(a[11], -h, h);         // k = 6
        a[13] = tw_const<DIR>(a[13], s1, c1);        // k = 3
        a[14] = tw_const<DIR>(a[14], -h, h);         // k = 6
        a[15] = tw_const<DIR>(a[15], -c1, -s1);      // k = 9
#pragma unroll
        for (int q = 0; q < 4; ++q) dft4<DIR>(a[4 * q], a[4 * q + 1], a[4 * q + 2], a[4 * q + 3]);
        // position 4*s1 + s2 holds X[s1 + 4*s2]: transpose the 4x4 register tile
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int j = i + 1; j < 4; ++j) { C t = a[4 * i + j]; a[4 * i + j] = a[4 * j + i]; a[4 * j + i] = t; }
    } else if constexpr (R == 32) {
        // R1 = 4 (over a), R2 = 8 (b): r = 8a + b
#pragma unroll
        for (int b = 0; b < 8; ++b) dft4<DIR>(a[b], a[8 + b], a[16 + b], a[24 + b]);
        // u[8*s1 + b] *= W32^(b*s1)
#pragma unroll
        for (int s1 = 1; s1 < 4; ++s1)
#pragma unroll
            for (int b = 1; b < 8; ++b) {
                const int k = b * s1;
                if (k == 8) a[8 * s1 + b] = mul_dir_i<DIR>(a[8 * s1 + b]);
                else a[8 * s1 + b] = tw_const<DIR>(a[8 * s1 + b], (T)cos32(k), (T)sin32(k));
            }
#pragma unroll
        for (int q = 0; q < 4; ++q)
            dft8r<DIR, T>(a[8 * q], a[8 * q + 1], a[8 * q + 2], a[8 * q + 3], a[8 * q + 4], a[8 * q + 5], a[8 * q + 6], a[8 * q + 7]);
        // position 8*s1 + s2 holds X[s1 + 4*s2]
        C o[32];
#pragma unroll
        for (int q = 0; q < 4; ++q)
#pragma unroll
            for (int s2 = 0; s2 < 8; ++s2) o[q + 4 * s2] = a[8 * q + s2];
#pragma unroll
        for (int i = 0; i < 32; ++i) a[i] = o[i];
    } else if constexpr (R == 10) {
        // R1 = 2 (over a), R2 = 5 (b): r = 5a + b
        const T C1 = (T)0.80901699437494742410, S1 = (T)0.58778525229247312917;   // (cos, sin)(2 pi / 10)
        const T C2 = (T)0.30901699437494742410, S2 = (T)0.95105651629515357212;   // k = 2
#pragma unroll
        for (int b = 0; b < 5; ++b) dft2<DIR>(a[b], a[5 + b]);
        // u[5*s1 + b] *= W10^(b*s1), s1 = 1
        a[6] = tw_const<DIR>(a[6], C1, S1);
        a[7] = tw_const<DIR>(a[7], C2, S2);
        a[8] = tw_const<DIR>(a[8], -C2, S2);        // k = 3: cos(108deg), sin(108deg)
        a[9] = tw_const<DIR>(a[9], -C1, S1);        // k = 4: cos(144deg), sin(144deg)
#pragma unroll
        for (int q = 0; q < 2; ++q) dft5<DIR, T>(a[5 * q], a[5 * q + 1], a[5 * q + 2], a[5 * q + 3], a[5 * q + 4]);
        // position 5*s1 + s2 holds X[s1 + 2*s2]
        C o[10];
#pragma unroll
        for (int q = 0; q < 2; ++q)
#pragma unroll
            for (int s2 = 0; s2 < 5; ++s2) o[q + 2 * s2] = a[5 * q + s2];
#pragma unroll
        for (int i = 0; i < 10; ++i) a[i] = o[i];
    } else if constexpr (R == 20) {
        // R1 = 4 (over a), R2 = 5 (b): r = 5a + b
#pragma unroll
        for (int b = 0; b < 5; ++b) dft4<DIR>(a[b], a[5 + b], a[10 + b], a[15 + b]);
        // u[5*s1 + b] *= W20^(b*s1); (cos, sin)(2 pi k / 20)
        const T C1 = (T)0.95105651629515357212, S1 = (T)0.30901699437494742410;   // k = 1
        const T C2 = (T)0.80901699437494742410, S2 = (T)0.58778525229247312917;   // k = 2
        const T C3 = (T)0.58778525229247312917, S3 = (T)0.80901699437494742410;   // k = 3
        const T C4 = (T)0.30901699437494742410, S4 = (T)0.95105651629515357212;   // k = 4
        a[6]  = tw_const<DIR>(a[6], C1, S1);         // s1=1,b=1: k=1
        a[7]  = tw_const<DIR>(a[7], C2, S2);         // k=2
        a[8]  = tw_const<DIR>(a[8], C3, S3);         // k=3
        a[9]  = tw_const<DIR>(a[9], C4, S4);         // k=4
        a[11] = tw_const<DIR>(a[11], C2, S2);        // s1=2,b=1: k=2
        a[12] = tw_const<DIR>(a[12], C4, S4);        // k=4
        a[13] = tw_const<DIR>(a[13], -S1, C1);       // k=6: cos(108deg) = -sin(18deg), sin(108deg) = cos(18deg)
        a[14] = tw_const<DIR>(a[14], -C2, S2);       // k=8: cos(144deg), sin(144deg)
        a[16] = tw_const<DIR>(a[16], C3, S3);        // s1=3,b=1: k=3
        a[17] = tw_const<DIR>(a[17], -S1, C1);       // k=6
        a[18] = tw_const<DIR>(a[18], -C1, S1);       // k=9: cos(162deg), sin(162deg)
        a[19] = tw_const<DIR>(a[19], -C2, -S2);      // k=12: cos(216deg), sin(216deg)
#pragma unroll
        for (int q = 0; q < 4; ++q) dft5<DIR, T>(a[5 * q], a[5 * q + 1], a[5 * q + 2], a[5 * q + 3], a[5 * q + 4]);
        // position 5*s1 + s2 holds X[s1 + 4*s2]
        C o[20];
#pragma unroll
        for (int q = 0; q < 4; ++q)
#pragma unroll
            for (int s2 = 0; s2 < 5; ++s2) o[q + 4 * s2] = a[5 * q + s2];
#pragma unroll
        for (int i = 0; i < 20; ++i) a[i] = o[i];
    } else {
        static_assert(R == 2, "unsupported radix");
    }
}

// ---------------------------------------------------------------- plans
// Elements per thread: float 32 (L >= 512) or 16, double 8, 5*2^k lengths 20.
#ifndef SGP_ROW_MINB
#define SGP_ROW_MINB 2        // resident CTAs per SM the row kernels are compiled for (register cap 128 at 2)
#endif
#ifndef SGP_ROW_E16
#define SGP_ROW_E16 0         // experiment: 16 elements per thread in the float row kernels (two warps per 2048-pixel row)
#endif
template <typename T> __host__ __device__ constexpr int fft_E(int L)
{
    return (L % 5 == 0) ? 20 : (sizeof(T) == 8 ? 8 : ((L >= 512 && !SGP_ROW_E16) ? 32 : 16));
}
// column kernel: a thread holds 32 elements only where that saves a pass (L = 512, 1024)
#ifndef SGP_COL_E32_ALL
#define SGP_COL_E32_ALL 0
#endif
#ifndef SGP_COL_E8_MIN
#define SGP_COL_E8_MIN (1 << 30)
#endif
template <typename T> __host__ __device__ constexpr int fft_E_col(int L)
{
    if (sizeof(T) == 4 && L % 5 != 0 && L >= SGP_COL_E8_MIN) return 8;
    return (L % 5 == 0) ? 20 : (sizeof(T) == 8 ? 8 : ((SGP_COL_E32_ALL ? L >= 512 : (L == 512 || L == 1024)) ? 32 : 16));
}
// radix of pass ip (0 = not a pass of this plan)
__host__ __device__ constexpr int plan_radix(int L, int E, int ip)
{
    if (E == 32) {
        switch (L) {
        case 512:  return ip == 0 ? 32 : ip == 1 ? 16 : 0;
        case 1024: return ip <= 1 ? 32 : 0;
        case 2048: return ip == 0 ? 32 : ip <= 2 ? 8 : 0;
        case 4096: return ip == 0 ? 32 : ip == 1 ? 16 : ip == 2 ? 8 : 0;
        }
    } else if (E == 16) {
        switch (L) {
        case 16:   return ip == 0 ? 16 : 0;
        case 32:   return ip == 0 ? 16 : ip == 1 ? 2 : 0;
        case 64:   return ip == 0 ? 16 : ip == 1 ? 4 : 0;
        case 128:  return ip == 0 ? 16 : ip == 1 ? 8 : 0;
        case 256:  return ip <= 1 ? 16 : 0;
        case 512:  return ip == 0 ? 16 : ip == 1 ? 8 : ip == 2 ? 4 : 0;
        case 1024: return ip <= 1 ? 16 : ip == 2 ? 4 : 0;
        case 2048: return ip <= 1 ? 16 : ip == 2 ? 8 : 0;
        case 4096: return ip <= 2 ? 16 : 0;
        }
    } else if (E == 8) {
        switch (L) {
        case 8:    return ip == 0 ? 8 : 0;
        case 16:   return ip == 0 ? 8 : ip == 1 ? 2 : 0;
        case 32:   return ip == 0 ? 8 : ip == 1 ? 4 : 0;
        case 64:   return ip <= 1 ? 8 : 0;
        case 128:  return ip == 0 ? 8 : ip <= 2 ? 4 : 0;
        case 256:  return ip <= 1 ? 8 : ip == 2 ? 4 : 0;
        case 512:  return ip <= 2 ? 8 : 0;
        case 1024: return ip <= 1 ? 8 : ip <= 3 ? 4 : 0;
        case 2048: return ip <= 2 ? 8 : ip == 3 ? 4 : 0;
        case 4096: return ip <= 3 ? 8 : 0;
        }
    } else if (E == 20) {
        switch (L) {
        case 20:   return ip == 0 ? 20 : 0;
        case 40:   return ip == 0 ? 20 : ip == 1 ? 2 : 0;
        case 80:   return ip == 0 ? 20 : ip == 1 ? 4 : 0;
        case 160:  return ip == 0 ? 20 : ip == 1 ? 4 : ip == 2 ? 2 : 0;
        case 320:  return ip == 0 ? 20 : ip <= 2 ? 4 : 0;
        case 640:  return ip == 0 ? 20 : ip <= 2 ? 4 : ip == 3 ? 2 : 0;
        case 1280: return ip == 0 ? 20 : ip <= 3 ? 4 : 0;
        // the other 2^a 5^b lengths: radix 20 first, then 20 / 10 / 5 / 4 / 2
        case 100:  return ip == 0 ? 20 : ip == 1 ? 5 : 0;
        case 200:  return ip == 0 ? 20 : ip == 1 ? 10 : 0;
        case 400:  return ip <= 1 ? 20 : 0;
        case 500:  return ip == 0 ? 20 : ip <= 2 ? 5 : 0;
        case 800:  return ip <= 1 ? 20 : ip == 2 ? 2 : 0;
        case 1000: return ip == 0 ? 20 : ip == 1 ? 10 : ip == 2 ? 5 : 0;
        case 1600: return ip <= 1 ? 20 : ip == 2 ? 4 : 0;
        case 2000: return ip <= 1 ? 20 : ip == 2 ? 5 : 0;
        case 2560: return ip == 0 ? 20 : ip <= 3 ? 4 : ip == 4 ? 2 : 0;
        case 3200: return ip <= 1 ? 20 : ip == 2 ? 4 : ip == 3 ? 2 : 0;
        case 4000: return ip <= 1 ? 20 : ip == 2 ? 10 : 0;
        }
    }
    return 0;
}
__host__ __device__ constexpr bool plan_ok(int L, int E) { return plan_radix(L, E, 0) != 0; }

// Twiddle tables.  Pass ip >= 1 of a plan (NS = product of the earlier radices, R = its radix) multiplies input r of
// butterfly j by exp(-2 pi i r (j mod NS) / (NS R)).  The table of a pass is stored as [r-1][j mod NS], so that the
// threads of a warp (consecutive j) read consecutive entries; the tables of the passes follow each other.
__host__ __device__ constexpr int plan_ns(int L, int E, int ip)
{
    int ns = 1;
    for (int i = 0; i < ip; ++i) ns *= plan_radix(L, E, i);
    return ns;
}
__host__ __device__ constexpr int tw_offset(int L, int E, int ip)      // start of the table of pass ip (ip >= 1)
{
    int off = 0;
    for (int i = 1; i < ip; ++i) off += (plan_radix(L, E, i) - 1) * plan_ns(L, E, i);
    return off;
}
__host__ __device__ constexpr int tw_total(int L, int E)
{
    int ip = 1;
    while (plan_radix(L, E, ip) != 0) ++ip;
    return tw_offset(L, E, ip) > 0 ? tw_offset(L, E, ip) : 1;
}

// shared-memory index padding: one extra slot every 2^PS elements (PS = 5 when the first pass is radix 32,
// else 4) turns the stride-R stores of the first pass into an odd stride, and keeps the reversed reads of the
// real<->complex untangling spread over the banks
__host__ __device__ constexpr int pad_shift(int E) { return E == 32 ? 5 : 4; }
template <int E> __host__ __device__ constexpr int fft_pad(int i) { return i + (i >> pad_shift(E)); }
__host__ __device__ constexpr int fft_padded_len(int L, int E) { return L + (L >> pad_shift(E)); }
// distance between the lines of two rows of a row-kernel CTA: even, so that every line starts on a 16-byte boundary (128-bit
// accesses of the epilogues, cp.async) also where the padded length is odd (L = 80, 400, 500, 2000)
__host__ __device__ constexpr int row_stride(int L, int E) { return (fft_padded_len(L, E) + 1) & ~1; }

// Threads that work on one row FFT of TF = L/E lanes.  A group must be synchronisable on its own: within a warp (a power
// of two <= 32) or whole warps (named barrier), so for the 5-smooth lengths (TF = 5, 10, 25, 40, 50, 100, ...) the group is
// padded to TFP threads; the lanes t >= TF repeat lane TF - 1 (same loads, same shared-memory traffic), take part in the
// barriers, and neither store to global memory nor contribute to a reduction.
__host__ __device__ constexpr int group_threads(int TF)
{
    if (TF <= 32) { int p = 1; while (p < TF) p *= 2; return p; }
    return (TF + 31) / 32 * 32;
}

// ---------------------------------------------------------------- synchronisation of the threads of one FFT
// SyncBlock: all threads of the CTA (column kernel: the columns of a tile are interleaved over the warps).
// SyncGroup<TF>: the TF threads of one row: __syncwarp when a warp holds whole rows, else a named barrier
// (id 1 + row slot, TF threads), so that the rows of a CTA never wait for each other.
struct SyncBlock { __device__ __forceinline__ void operator()() const { __syncthreads(); } };
template <int TF> struct SyncGroup {
    int id;
    __device__ __forceinline__ void operator()() const
    {
        if constexpr (TF <= 32) __syncwarp();
        else asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(TF) : "memory");
    }
};

// All passes of one FFT.  sm points at element 0 of this FFT's shared-memory line; consecutive
// elements are `cs` apart (1 for a row FFT; C for a column FFT stored as [element][column]).
// tw = the per-pass twiddle tables of this plan (see above).  Every exchange is bracketed sync / store / sync / load, so shared memory
// the caller used before the call is safe to reuse, and on return nobody is writing it.
// TWS: the tables sit in shared memory (copied there by the caller), else in global memory (read-only path)
template <typename T, int L, int E, int DIR, int IP, int NS, bool TWS, bool TWP, typename SYNC>
__device__ __forceinline__ void fft_passes(cx<T> (&v)[E], cx<T> *__restrict__ sm, const int cs, const int t,
                                           const cx<T> *__restrict__ tw, const SYNC &sync)
{
    using C = cx<T>;
    constexpr int R = plan_radix(L, E, IP);
    static_assert(R > 0 && E % R == 0, "bad plan");
    constexpr int B = E / R;
    constexpr int TF = L / E;
    constexpr bool LAST = (NS * R == L);
    int j0s[B];
#pragma unroll
    for (int b = 0; b < B; ++b) {
        C a[R];
#pragma unroll
        for (int r = 0; r < R; ++r) a[r] = v[b + r * B];
        const int j = t + b * TF;
        if constexpr (NS > 1) {
            const int jm = j % NS;                       // NS is a compile-time constant
            const C *twp = tw + tw_offset(L, E, IP) + jm;
            if constexpr (TWP && (R == 8 || R == 16 || R == 32)) {
                // TWP: the R - 1 twiddles w^r, w = exp(-2 pi i jm / (NS R)), from H - 1 + R/H - 1 table entries and ONE product each:
                // w^(aH + b) = w^(aH) w^b with w^1 .. w^(H-1) and w^H, w^2H, ... loaded (H = 4; 2 for radix 8): 6 loads + 9 products
                // instead of 15 loads at radix 16, 10 + 21 instead of 31 at radix 32, 4 + 3 instead of 7 at radix 8.  Every value is
                // a table entry or the product of two, so its error stays at two table roundings plus one product.  (Powers of the
                // single entry w^1 -- one load -- are faster still and far too noisy: the rounding of w^1 comes back r times in w^r.)
                // An option of the float kernels (col.cuh: SGP_COL_TWP, row_fwd.cuh: SGP_ROW_TWP), off by default.
                constexpr int H = R >= 16 ? 4 : 2;
                auto twmul = [](C x, C w) { return (DIR < 0) ? cmul(x, w) : cmulc(x, w); };
                C wl[H];
#pragma unroll
                for (int lo = 1; lo < H; ++lo) { wl[lo] = __ldg(&twp[(lo - 1) * NS]); a[lo] = twmul(a[lo], wl[lo]); }
#pragma unroll
                for (int hi = 1; hi < R / H; ++hi) {
                    const C wh = __ldg(&twp[(hi * H - 1) * NS]);
                    a[hi * H] = twmul(a[hi * H], wh);
#pragma unroll
                    for (int lo = 1; lo < H; ++lo) a[hi * H + lo] = twmul(a[hi * H + lo], cmul(wh, wl[lo]));
                }
            } else {
#pragma unroll
                for (int r = 1; r < R; ++r) {
                    C w = TWS ? twp[(r - 1) * NS] : __ldg(&twp[(r - 1) * NS]);
                    a[r] = (DIR < 0) ? cmul(a[r], w) : cmulc(a[r], w);
                }
            }
            j0s[b] = (j / NS) * (NS * R) + jm;
        } else {
            j0s[b] = j * R;
        }
        dft<R, DIR, T>(a);
#pragma unroll
        for (int s = 0; s < R; ++s) v[b + s * B] = a[s];
    }
    if constexpr (!LAST) {
        sync();
#pragma unroll
        for (int b = 0; b < B; ++b)
#pragma unroll
            for (int s = 0; s < R; ++s) sm[fft_pad<E>(j0s[b] + s * NS) * cs] = v[b + s * B];
        sync();
#pragma unroll
        for (int e = 0; e < E; ++e) v[e] = sm[fft_pad<E>(t + TF * e) * cs];
        fft_passes<T, L, E, DIR, IP + 1, NS * R, TWS, TWP>(v, sm, cs, t, tw, sync);
    }
}

template <typename T, int L, int E, int DIR, bool TWS = false, bool TWP = false, typename SYNC>
__device__ __forceinline__ void fft_block(cx<T> (&v)[E], cx<T> *sm, int cs, int t, const cx<T> *tw, const SYNC &sync)
{
    fft_passes<T, L, E, DIR, 0, 1, TWS, TWP>(v, sm, cs, t, tw, sync);
}

// Twiddle tables in shared memory.  The pass tables of a transform are read (R - 1)/R times per element and pass -- as
// often as the exchange buffer -- and as global loads they miss a good part of the time in what the shared-memory
// carve-out leaves of the L1 (ncu, 2048^2: 28 % of the column kernel's twiddle sectors, 200 KB carve-out), each miss a trip
// to L2 that the 4 warps per scheduler cannot hide: "long scoreboard" was the top stall of every FFT kernel.
#ifndef SGP_TW_SMEM
#define SGP_TW_SMEM 0      // measured at 2048^2 (round 2): every FFT kernel 0.5-2 us SLOWER with the tables in shared memory -- off
#endif
template <typename C>
__device__ __forceinline__ void copy_table_to_smem(C *dst, const C *__restrict__ src, int count, int tid, int nthr)
{
    for (int i = tid; i < count; i += nthr) dst[i] = __ldg(&src[i]);
}

}  // namespace sgpk
