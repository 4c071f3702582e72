// codelets.cuh -- register-resident radix-R complex fp64 DFT butterflies (R = 2, 3, 4, 5, 6, 8, 15, 16).
//
// Building blocks of the hand-written FFT passes (BASELINE.json north_star (1): "radix-2/3/4/8/16
// stages").  Each codelet transforms R values held in registers IN PLACE and leaves them in NATURAL
// order:  v[k] <- sum_a v[a] exp(-/+ 2 pi i a k / R)   (INV = false: minus sign, forward DFT;
// INV = true: plus sign, unnormalised inverse).  Register indices are compile-time after unrolling, so
// "natural order" costs no data movement.
#pragma once
#include <cuda_runtime.h>

namespace ptfock {

typedef double2 cd;

#define PTF_DEV __device__ __forceinline__

PTF_DEV cd cadd(cd a, cd b) { return make_double2(a.x + b.x, a.y + b.y); }
PTF_DEV cd csub(cd a, cd b) { return make_double2(a.x - b.x, a.y - b.y); }
PTF_DEV cd cmul(cd a, cd b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
// a * conj(b)
PTF_DEV cd cmulc(cd a, cd b) { return make_double2(a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y); }
PTF_DEV cd cconj(cd a) { return make_double2(a.x, -a.y); }
PTF_DEV cd cscale(cd a, double s) { return make_double2(a.x * s, a.y * s); }

// multiply by exp(-/+ i pi/2) = -/+ i
template <bool INV> PTF_DEV cd mul_mi(cd a) { return INV ? make_double2(-a.y, a.x) : make_double2(a.y, -a.x); }
// multiply by a forward-sign twiddle w (INV: by conj(w))
template <bool INV> PTF_DEV cd twmul(cd a, cd w) { return INV ? cmulc(a, w) : cmul(a, w); }

constexpr double kSqrtHalf = 0.70710678118654752440084436210485;
constexpr double kCosPi8 = 0.92387953251128675612818318939679;
constexpr double kSinPi8 = 0.38268343236508977172845998403040;
constexpr double kSin2Pi3 = 0.86602540378443864676372317075294;

template <int R, bool INV> struct DFT;

template <bool INV> struct DFT<1, INV> {
    static PTF_DEV void run(cd (&)[1]) {}
};

template <bool INV> struct DFT<2, INV> {
    static PTF_DEV void run(cd (&v)[2]) {
        cd a = v[0], b = v[1];
        v[0] = cadd(a, b);
        v[1] = csub(a, b);
    }
};

template <bool INV> struct DFT<3, INV> {
    static PTF_DEV void run(cd (&v)[3]) {
        cd t = cadd(v[1], v[2]);
        cd d = csub(v[1], v[2]);
        cd m = make_double2(v[0].x - 0.5 * t.x, v[0].y - 0.5 * t.y);
        // u = (-/+ i) sin(2pi/3) d
        cd u = mul_mi<INV>(cscale(d, kSin2Pi3));
        v[0] = cadd(v[0], t);
        v[1] = cadd(m, u);
        v[2] = csub(m, u);
    }
};

// radix 5 (the paper's own grid 60 x 90 x 120, needs the factor 5)
constexpr double kCos2Pi5 = 0.30901699437494742410229341718282;
constexpr double kCos4Pi5 = -0.80901699437494742410229341718282;
constexpr double kSin2Pi5 = 0.95105651629515357211643933337938;
constexpr double kSin4Pi5 = 0.58778525229247312916870595463907;

template <bool INV> struct DFT<5, INV> {
    static PTF_DEV void run(cd &x0, cd &x1, cd &x2, cd &x3, cd &x4) {
        const cd t1 = cadd(x1, x4), t2 = cadd(x2, x3), t3 = csub(x1, x4), t4 = csub(x2, x3);
        const cd m1 = make_double2(x0.x + kCos2Pi5 * t1.x + kCos4Pi5 * t2.x, x0.y + kCos2Pi5 * t1.y + kCos4Pi5 * t2.y);
        const cd m2 = make_double2(x0.x + kCos4Pi5 * t1.x + kCos2Pi5 * t2.x, x0.y + kCos4Pi5 * t1.y + kCos2Pi5 * t2.y);
        // s1 = sin(2pi/5) t3 + sin(4pi/5) t4,  s2 = sin(4pi/5) t3 - sin(2pi/5) t4;  X1,4 = m1 -/+ i s1,  X2,3 = m2 -/+ i s2
        const cd s1 = mul_mi<INV>(make_double2(kSin2Pi5 * t3.x + kSin4Pi5 * t4.x, kSin2Pi5 * t3.y + kSin4Pi5 * t4.y));
        const cd s2 = mul_mi<INV>(make_double2(kSin4Pi5 * t3.x - kSin2Pi5 * t4.x, kSin4Pi5 * t3.y - kSin2Pi5 * t4.y));
        x0 = make_double2(x0.x + t1.x + t2.x, x0.y + t1.y + t2.y);
        x1 = cadd(m1, s1);
        x4 = csub(m1, s1);
        x2 = cadd(m2, s2);
        x3 = csub(m2, s2);
    }
    static PTF_DEV void run(cd (&v)[5]) { run(v[0], v[1], v[2], v[3], v[4]); }
};

// radix 6 = 2 x 3 and radix 15 = 3 x 5 by the prime-factor (Good-Thomas) map: coprime factors need no twiddles.
//   n = (N2 n1 + N1 n2) mod N,  k = (c1 k1 + c2 k2) mod N  with c1 = 1 mod N1, 0 mod N2 and c2 = 0 mod N1, 1 mod N2.
template <bool INV> struct DFT<6, INV> {
    static PTF_DEV void run(cd (&v)[6]) {
        // n = 3 n1 + 2 n2 (n1 < 2, n2 < 3); k = 3 k1 + 4 k2 mod 6
        cd a[2][3];
#pragma unroll
        for (int n1 = 0; n1 < 2; ++n1)
#pragma unroll
            for (int n2 = 0; n2 < 3; ++n2) a[n1][n2] = v[(3 * n1 + 2 * n2) % 6];
#pragma unroll
        for (int n1 = 0; n1 < 2; ++n1) DFT<3, INV>::run(a[n1]);
#pragma unroll
        for (int k2 = 0; k2 < 3; ++k2) {
            const cd e = a[0][k2], o = a[1][k2];
            v[(4 * k2) % 6] = cadd(e, o);
            v[(3 + 4 * k2) % 6] = csub(e, o);
        }
    }
};

template <bool INV> struct DFT<15, INV> {
    static PTF_DEV void run(cd (&v)[15]) {
        // n = 5 n1 + 3 n2 (n1 < 3, n2 < 5); k = 10 k1 + 6 k2 mod 15
        cd a[3][5];
#pragma unroll
        for (int n1 = 0; n1 < 3; ++n1)
#pragma unroll
            for (int n2 = 0; n2 < 5; ++n2) a[n1][n2] = v[(5 * n1 + 3 * n2) % 15];
#pragma unroll
        for (int n1 = 0; n1 < 3; ++n1) DFT<5, INV>::run(a[n1]);
#pragma unroll
        for (int k2 = 0; k2 < 5; ++k2) {
            cd c[3] = { a[0][k2], a[1][k2], a[2][k2] };
            DFT<3, INV>::run(c);
#pragma unroll
            for (int k1 = 0; k1 < 3; ++k1) v[(10 * k1 + 6 * k2) % 15] = c[k1];
        }
    }
};

// radix 24 = 3 x 8 by the same map: n = 8 n1 + 3 n2 (n1 < 3, n2 < 8); k = 16 k1 + 9 k2 mod 24.
// (Declared after DFT<8>: see below.)

template <bool INV> struct DFT<4, INV> {
    static PTF_DEV void run(cd &a0, cd &a1, cd &a2, cd &a3) {
        cd t0 = cadd(a0, a2), t1 = csub(a0, a2);
        cd t2 = cadd(a1, a3), t3 = mul_mi<INV>(csub(a1, a3));
        a0 = cadd(t0, t2);
        a2 = csub(t0, t2);
        a1 = cadd(t1, t3);
        a3 = csub(t1, t3);
    }
    static PTF_DEV void run(cd (&v)[4]) { run(v[0], v[1], v[2], v[3]); }
};

template <bool INV> struct DFT<8, INV> {
    static PTF_DEV void run(cd (&v)[8]) {
        // decimation in time: even / odd halves, then the w8^k combine
        DFT<4, INV>::run(v[0], v[2], v[4], v[6]);   // E[0..3] in v[0], v[2], v[4], v[6]
        DFT<4, INV>::run(v[1], v[3], v[5], v[7]);   // O[0..3] in v[1], v[3], v[5], v[7]
        cd o0 = v[1];
        // w8^1 = (1 -/+ i)/sqrt2 ; w8^2 = -/+ i ; w8^3 = (-1 -/+ i)/sqrt2
        cd o1 = INV ? make_double2((v[3].x - v[3].y) * kSqrtHalf, (v[3].x + v[3].y) * kSqrtHalf)
                    : make_double2((v[3].x + v[3].y) * kSqrtHalf, (v[3].y - v[3].x) * kSqrtHalf);
        cd o2 = mul_mi<INV>(v[5]);
        cd o3 = INV ? make_double2(-(v[7].x + v[7].y) * kSqrtHalf, (v[7].x - v[7].y) * kSqrtHalf)
                    : make_double2((v[7].y - v[7].x) * kSqrtHalf, -(v[7].x + v[7].y) * kSqrtHalf);
        cd e0 = v[0], e1 = v[2], e2 = v[4], e3 = v[6];
        v[0] = cadd(e0, o0); v[4] = csub(e0, o0);
        v[1] = cadd(e1, o1); v[5] = csub(e1, o1);
        v[2] = cadd(e2, o2); v[6] = csub(e2, o2);
        v[3] = cadd(e3, o3); v[7] = csub(e3, o3);
    }
};

template <bool INV> struct DFT<24, INV> {
    static PTF_DEV void run(cd (&v)[24]) {
        cd a[3][8];
#pragma unroll
        for (int n1 = 0; n1 < 3; ++n1)
#pragma unroll
            for (int n2 = 0; n2 < 8; ++n2) a[n1][n2] = v[(8 * n1 + 3 * n2) % 24];
#pragma unroll
        for (int n1 = 0; n1 < 3; ++n1) DFT<8, INV>::run(a[n1]);
#pragma unroll
        for (int k2 = 0; k2 < 8; ++k2) {
            cd c[3] = { a[0][k2], a[1][k2], a[2][k2] };
            DFT<3, INV>::run(c);
#pragma unroll
            for (int k1 = 0; k1 < 3; ++k1) v[(16 * k1 + 9 * k2) % 24] = c[k1];
        }
    }
};

template <bool INV> struct DFT<16, INV> {
    // first half: 16 = 4 x 4, x = 4a + b.  DFT over a for each b, then the twiddles w16^(b k1).
    // Afterwards v[4 k1 + b] = y[k1][b] and X[k1 + 4 k2] = DFT4 over b of y[k1][.].
    static PTF_DEV void first_half(cd (&v)[16]) {
#pragma unroll
        for (int b = 0; b < 4; ++b) DFT<4, INV>::run(v[b], v[4 + b], v[8 + b], v[12 + b]);
        const cd w1 = make_double2(kCosPi8, -kSinPi8);        // w16^1 (forward sign)
        const cd w2 = make_double2(kSqrtHalf, -kSqrtHalf);    // w16^2
        const cd w3 = make_double2(kSinPi8, -kCosPi8);        // w16^3
        const cd w6 = make_double2(-kSqrtHalf, -kSqrtHalf);   // w16^6
        const cd w9 = make_double2(-kCosPi8, kSinPi8);        // w16^9
        v[4 + 1] = twmul<INV>(v[4 + 1], w1);
        v[4 + 2] = twmul<INV>(v[4 + 2], w2);
        v[4 + 3] = twmul<INV>(v[4 + 3], w3);
        v[8 + 1] = twmul<INV>(v[8 + 1], w2);
        v[8 + 2] = mul_mi<INV>(v[8 + 2]);                      // w16^4 = -/+ i
        v[8 + 3] = twmul<INV>(v[8 + 3], w6);
        v[12 + 1] = twmul<INV>(v[12 + 1], w3);
        v[12 + 2] = twmul<INV>(v[12 + 2], w6);
        v[12 + 3] = twmul<INV>(v[12 + 3], w9);
    }
    // second half for one k1: on return v[4 k1 + k2] = X[k1 + 4 k2]
    static PTF_DEV void second_half(cd (&v)[16], int k1) {
        DFT<4, INV>::run(v[4 * k1], v[4 * k1 + 1], v[4 * k1 + 2], v[4 * k1 + 3]);
    }
    static PTF_DEV void run(cd (&v)[16]) {
        first_half(v);
#pragma unroll
        for (int k1 = 0; k1 < 4; ++k1) second_half(v, k1);
        // v[4 k1 + k2] holds X[k1 + 4 k2]: transpose the 4x4 register tile (free: renaming)
#pragma unroll
        for (int k1 = 0; k1 < 4; ++k1)
#pragma unroll
            for (int k2 = k1 + 1; k2 < 4; ++k2) {
                cd t = v[4 * k1 + k2];
                v[4 * k1 + k2] = v[4 * k2 + k1];
                v[4 * k2 + k1] = t;
            }
    }
};

}  // namespace ptfock
