// fft_codelets.cuh -- in-register complex128 DFT codelets for radices dividing 48 (2,3,4,6,8,12,16,24).
//
// Every index below is a compile-time constant after unrolling, so the arrays live in registers and the butterfly
// twiddles fold into immediates.  DIR = -1: forward (e^{-i...}), DIR = +1: inverse (unnormalised).
#pragma once
#include <cuda_runtime.h>
#include "twiddle48.h"

namespace tdh {

typedef double2 cd;   // .x = re, .y = im

__device__ __forceinline__ cd cmake(double re, double im) { return make_double2(re, im); }
__device__ __forceinline__ cd cadd(cd a, cd b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ cd csub(cd a, cd b) { return make_double2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ cd cscale(cd a, double s) { return make_double2(a.x * s, a.y * s); }
__device__ __forceinline__ cd cmul(cd a, cd b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
// a * conj(b)
__device__ __forceinline__ cd cmulc(cd a, cd b) { return make_double2(a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y); }
__device__ __forceinline__ cd cfma(cd a, cd b, cd c) {   // a*b + c
    return make_double2(fma(a.x, b.x, fma(-a.y, b.y, c.x)), fma(a.x, b.y, fma(a.y, b.x, c.y)));
}
// multiply by +i / -i
__device__ __forceinline__ cd cmuli(cd a) { return make_double2(-a.y, a.x); }
__device__ __forceinline__ cd cmulni(cd a) { return make_double2(a.y, -a.x); }

// cos / sin of 2 pi k / 48 from the generated quarter-wave table
__host__ __device__ constexpr double cos48(int k) {
    constexpr double tab[13] = TDH_COS48_TABLE;
    k = ((k % 48) + 48) % 48;
    if (k > 24) k = 48 - k;            // cos(2pi - x) = cos x
    return k > 12 ? -tab[24 - k] : tab[k];
}
__host__ __device__ constexpr double sin48(int k) { return cos48(k - 12); }

// a * exp(DIR * 2 pi i * NUM / DEN), all compile time; DEN must divide 48.
template <int NUM, int DEN, int DIR>
__device__ __forceinline__ cd twmul(cd a) {
    static_assert(48 % DEN == 0, "twiddle denominator must divide 48");
    constexpr int K0 = (((48 / DEN) * NUM) % 48 + 48) % 48;
    constexpr int K = DIR > 0 ? K0 : (48 - K0) % 48;   // angle 2 pi K / 48, counter-clockwise
    if constexpr (K == 0) return a;
    else if constexpr (K == 12) return cmuli(a);
    else if constexpr (K == 24) return make_double2(-a.x, -a.y);
    else if constexpr (K == 36) return cmulni(a);
    else if constexpr (K == 6) { constexpr double h = cos48(6); return make_double2((a.x - a.y) * h, (a.x + a.y) * h); }
    else if constexpr (K == 18) { constexpr double h = cos48(6); return make_double2((-a.x - a.y) * h, (a.x - a.y) * h); }
    else if constexpr (K == 30) { constexpr double h = cos48(6); return make_double2((a.y - a.x) * h, (-a.x - a.y) * h); }
    else if constexpr (K == 42) { constexpr double h = cos48(6); return make_double2((a.x + a.y) * h, (a.y - a.x) * h); }
    else {
        constexpr double c = cos48(K), s = sin48(K);
        return make_double2(a.x * c - a.y * s, a.x * s + a.y * c);
    }
}

template <int R, int DIR> struct Dft;

template <int DIR> struct Dft<1, DIR> {
    static __device__ __forceinline__ void run(cd (&)[1]) {}
};

template <int DIR> struct Dft<2, DIR> {
    static __device__ __forceinline__ void run(cd (&x)[2]) {
        cd a = x[0], b = x[1];
        x[0] = cadd(a, b);
        x[1] = csub(a, b);
    }
};

template <int DIR> struct Dft<3, DIR> {
    static __device__ __forceinline__ void run(cd (&x)[3]) {
        constexpr double s3 = cos48(4) * DIR;   // +-sqrt(3)/2
        cd a = x[0], b = x[1], c = x[2];
        cd t1 = cadd(b, c);
        cd t2 = make_double2(a.x - 0.5 * t1.x, a.y - 0.5 * t1.y);
        cd d = csub(b, c);
        cd t3 = make_double2(-s3 * d.y, s3 * d.x);   // i * DIR * sqrt(3)/2 * (b - c)
        x[0] = cadd(a, t1);
        x[1] = cadd(t2, t3);
        x[2] = csub(t2, t3);
    }
};

template <int DIR> struct Dft<4, DIR> {
    static __device__ __forceinline__ void run(cd (&x)[4]) {
        cd t0 = cadd(x[0], x[2]), t1 = csub(x[0], x[2]);
        cd t2 = cadd(x[1], x[3]), d = csub(x[1], x[3]);
        cd t3 = DIR > 0 ? cmuli(d) : cmulni(d);      // exp(DIR i pi/2) (b - d)
        x[0] = cadd(t0, t2);
        x[1] = cadd(t1, t3);
        x[2] = csub(t0, t2);
        x[3] = csub(t1, t3);
    }
};

// split R = RA * RB: first RB transforms of length RA on stride RB, twiddle, then RA transforms of length RB.
template <int R> struct Split {
    static constexpr int RA = (R % 4 == 0 && R > 4) ? 4 : ((R % 3 == 0 && R > 3) ? 3 : 2);
    static constexpr int RB = R / RA;
};

template <int RA, int RB, int DIR, int K1, int J2>
__device__ __forceinline__ void tw_row(cd (&s)[RB][RA]) {
    if constexpr (J2 < RB) {
        s[J2][K1] = twmul<J2 * K1, RA * RB, DIR>(s[J2][K1]);
        tw_row<RA, RB, DIR, K1, J2 + 1>(s);
    }
}
template <int RA, int RB, int DIR, int K1>
__device__ __forceinline__ void tw_all(cd (&s)[RB][RA]) {
    if constexpr (K1 < RA) {
        tw_row<RA, RB, DIR, K1, 1>(s);
        tw_all<RA, RB, DIR, K1 + 1>(s);
    }
}

template <int R, int DIR> struct Dft {
    static constexpr int RA = Split<R>::RA, RB = Split<R>::RB;
    static __device__ __forceinline__ void run(cd (&x)[R]) {
        cd s[RB][RA];
#pragma unroll
        for (int j2 = 0; j2 < RB; ++j2) {
#pragma unroll
            for (int j1 = 0; j1 < RA; ++j1) s[j2][j1] = x[RB * j1 + j2];
            Dft<RA, DIR>::run(s[j2]);
        }
        tw_all<RA, RB, DIR, 1>(s);
#pragma unroll
        for (int k1 = 0; k1 < RA; ++k1) {
            cd t[RB];
#pragma unroll
            for (int j2 = 0; j2 < RB; ++j2) t[j2] = s[j2][k1];
            Dft<RB, DIR>::run(t);
#pragma unroll
            for (int k2 = 0; k2 < RB; ++k2) x[k1 + RA * k2] = t[k2];
        }
    }
};

// Two-stage factorisation of a full axis length N = R1 * R2 (first stage radix R1 on stride R2).
template <int N> struct Fact;
template <> struct Fact<16> { static constexpr int R1 = 4, R2 = 4; };
template <> struct Fact<32> { static constexpr int R1 = 8, R2 = 4; };
template <> struct Fact<48> { static constexpr int R1 = 8, R2 = 6; };
template <> struct Fact<64> { static constexpr int R1 = 8, R2 = 8; };
template <> struct Fact<96> { static constexpr int R1 = 12, R2 = 8; };
// The plane kernels keep R1 - 1 twiddles in registers, so they prefer the smaller first radix for 96.
template <int N> struct FactP : Fact<N> {};
template <> struct FactP<96> { static constexpr int R1 = 8, R2 = 12; };

}  // namespace tdh
