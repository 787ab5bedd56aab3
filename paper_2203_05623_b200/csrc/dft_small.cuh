// In-register DFT codelets of size R in {2,3,4,6,8,9,12,16} on complex<T>, sign template (+1: exp(+i..), -1: exp(-i..)).
// Used by the sphere-pruned 3D FFT.  Fully unrolled; twiddles are compile-time literals (dft_consts.h).
#pragma once
#include "dft_consts.h"
#ifndef WHD
#define WHD __host__ __device__ __forceinline__
#endif

template <typename T>
struct alignas(2 * sizeof(T)) cx {      // 16-byte (f64) / 8-byte (f32) aligned: one LDS.128 / LDG.128 per element
    T x, y;
};
template <typename T> WHD cx<T> mk(T a, T b) { cx<T> r; r.x = a; r.y = b; return r; }
template <typename T> WHD cx<T> operator+(cx<T> a, cx<T> b) { return mk<T>(a.x + b.x, a.y + b.y); }
template <typename T> WHD cx<T> operator-(cx<T> a, cx<T> b) { return mk<T>(a.x - b.x, a.y - b.y); }
template <typename T> WHD cx<T> cmul(cx<T> a, cx<T> b) {
    return mk<T>(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
template <typename T> WHD cx<T> cmulc(cx<T> a, cx<T> b) {   // a * conj(b)
    return mk<T>(a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y);
}
template <typename T> WHD cx<T> cconj(cx<T> a) { return mk<T>(a.x, -a.y); }
// multiply by (SIGN * i)
template <typename T, int SIGN> WHD cx<T> mul_i(cx<T> a) {
    return SIGN > 0 ? mk<T>(-a.y, a.x) : mk<T>(a.y, -a.x);
}

template <int R> __host__ __device__ constexpr double dft_cos(int m) {
    return R == 6 ? dft_cos_6(m % 6) : R == 8 ? dft_cos_8(m % 8) : R == 9 ? dft_cos_9(m % 9)
         : R == 12 ? dft_cos_12(m % 12) : dft_cos_16(m % 16);
}
template <int R> __host__ __device__ constexpr double dft_sin(int m) {
    return R == 6 ? dft_sin_6(m % 6) : R == 8 ? dft_sin_8(m % 8) : R == 9 ? dft_sin_9(m % 9)
         : R == 12 ? dft_sin_12(m % 12) : dft_sin_16(m % 16);
}

// multiply a by exp(SIGN * 2 pi i m / R), m compile-time after unrolling; trivial cases cost no multiplies
template <typename T, int R, int SIGN> WHD cx<T> tw_small(cx<T> a, int m) {
    m = m % R;
    if (m == 0) return a;
    if (4 * m == R) return mul_i<T, SIGN>(a);
    if (2 * m == R) return mk<T>(-a.x, -a.y);
    if (4 * m == 3 * R) return mul_i<T, -SIGN>(a);
    if (8 * m == R || 8 * m == 3 * R || 8 * m == 5 * R || 8 * m == 7 * R) {
        const T h = (T)0.70710678118654752440;
        // exp(i s pi/4 * odd)
        const T c = (8 * m == R || 8 * m == 7 * R) ? h : -h;
        const T s0 = (8 * m == R || 8 * m == 3 * R) ? h : -h;
        const T s = SIGN > 0 ? s0 : -s0;
        // (a.x + i a.y)(c + i s), |c| = |s| = h
        const T px = a.x * h, py = a.y * h;
        const T rx = (c > 0 ? px : -px) - (s > 0 ? py : -py);
        const T ry = (s > 0 ? px : -px) + (c > 0 ? py : -py);
        return mk<T>(rx, ry);
    }
    const T c = (T)dft_cos<R>(m);
    const T s = (T)(SIGN > 0 ? dft_sin<R>(m) : -dft_sin<R>(m));
    return mk<T>(a.x * c - a.y * s, a.x * s + a.y * c);
}

template <typename T, int R, int SIGN> struct Dft;

template <typename T, int SIGN> struct Dft<T, 2, SIGN> {
    static WHD void run(cx<T> (&v)[2]) {
        cx<T> a = v[0] + v[1], b = v[0] - v[1];
        v[0] = a; v[1] = b;
    }
};
template <typename T, int SIGN> struct Dft<T, 3, SIGN> {
    static WHD void run(cx<T> (&v)[3]) {
        // 12 FP64 instructions: 6 adds, 2 + 4 fused multiply-adds (the sqrt(3)/2 rotation is folded into the last stage)
        const T s3 = SIGN > 0 ? (T)0.86602540378443864676 : (T)-0.86602540378443864676;
        const cx<T> t = v[1] + v[2];
        const cx<T> d = v[1] - v[2];
        const cx<T> m1 = mk<T>(v[0].x - (T)0.5 * t.x, v[0].y - (T)0.5 * t.y);
        v[0] = v[0] + t;
        // m2 = i * SIGN * (sqrt3/2) d = (-s3 d.y, s3 d.x)
        v[1] = mk<T>(m1.x - s3 * d.y, m1.y + s3 * d.x);
        v[2] = mk<T>(m1.x + s3 * d.y, m1.y - s3 * d.x);
    }
};
template <typename T, int SIGN> struct Dft<T, 4, SIGN> {
    static WHD void run(cx<T> (&v)[4]) {
        cx<T> a = v[0] + v[2], b = v[0] - v[2];
        cx<T> c = v[1] + v[3], d = mul_i<T, SIGN>(v[1] - v[3]);
        v[0] = a + c; v[2] = a - c;
        v[1] = b + d; v[3] = b - d;
    }
};

// Cooley-Tukey composite R = A*B in registers: input n = B a + b, output k = ka + A kb.
template <typename T, int A, int B, int SIGN> struct DftCT {
    static WHD void run(cx<T> (&v)[A * B]) {
        constexpr int R = A * B;
        cx<T> t[B][A];
#pragma unroll
        for (int b = 0; b < B; ++b) {
            cx<T> u[A];
#pragma unroll
            for (int a = 0; a < A; ++a) u[a] = v[B * a + b];
            Dft<T, A, SIGN>::run(u);
#pragma unroll
            for (int ka = 0; ka < A; ++ka) t[b][ka] = tw_small<T, R, SIGN>(u[ka], b * ka);
        }
#pragma unroll
        for (int ka = 0; ka < A; ++ka) {
            cx<T> s[B];
#pragma unroll
            for (int b = 0; b < B; ++b) s[b] = t[b][ka];
            Dft<T, B, SIGN>::run(s);
#pragma unroll
            for (int kb = 0; kb < B; ++kb) v[ka + A * kb] = s[kb];
        }
    }
};
template <typename T, int SIGN> struct Dft<T, 6, SIGN>  { static WHD void run(cx<T> (&v)[6])  { DftCT<T, 2, 3, SIGN>::run(v); } };
template <typename T, int SIGN> struct Dft<T, 8, SIGN>  { static WHD void run(cx<T> (&v)[8])  { DftCT<T, 2, 4, SIGN>::run(v); } };
template <typename T, int SIGN> struct Dft<T, 9, SIGN>  { static WHD void run(cx<T> (&v)[9])  { DftCT<T, 3, 3, SIGN>::run(v); } };
template <typename T, int SIGN> struct Dft<T, 12, SIGN> { static WHD void run(cx<T> (&v)[12]) { DftCT<T, 3, 4, SIGN>::run(v); } };
template <typename T, int SIGN> struct Dft<T, 16, SIGN> { static WHD void run(cx<T> (&v)[16]) { DftCT<T, 4, 4, SIGN>::run(v); } };
