// fft_radix.cuh -- register-level building blocks: complex helpers, compile-time twiddles and a
// fully unrolled in-register DFT of any length R = 2^a * 3^b * 5^c * 7^d (R <= 48 used).
//
// The transform implemented is the 1D DFT of Eq. (1)/(2) of the paper:
//   X[k] = sum_j x[j] exp(DIR * 2 pi i j k / R),  DIR = -1 forward, +1 inverse (unnormalised).
// Everything here is hand-written for sm_100a; no cuFFT, no library code.
#pragma once
#include <cuda_runtime.h>

namespace fft3d {

template <typename T> struct cx_sel;
template <> struct cx_sel<float>  { using type = float2; };
template <> struct cx_sel<double> { using type = double2; };
template <typename T> using cx = typename cx_sel<T>::type;

template <typename T> __host__ __device__ __forceinline__ cx<T> mk(T a, T b) { cx<T> r; r.x = a; r.y = b; return r; }
template <typename C> __device__ __forceinline__ C cadd(C a, C b) { C r; r.x = a.x + b.x; r.y = a.y + b.y; return r; }
template <typename C> __device__ __forceinline__ C csub(C a, C b) { C r; r.x = a.x - b.x; r.y = a.y - b.y; return r; }
template <typename C> __device__ __forceinline__ C cmul(C a, C b) {
    C r; r.x = a.x * b.x - a.y * b.y; r.y = a.x * b.y + a.y * b.x; return r;
}
template <typename C> __device__ __forceinline__ C cconj(C a) { C r; r.x = a.x; r.y = -a.y; return r; }
// fp32: Blackwell's packed f32x2 arithmetic (FADD2 / FMUL2 / FFMA2: one issue slot per complex operation; the
// swap / broadcast / per-half negation of the operands are free operand modifiers in SASS)
#ifdef __CUDA_ARCH__
__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return __fadd2_rn(a, make_float2(-b.x, -b.y)); }
__device__ __forceinline__ float2 cmul(float2 a, float2 w) {
    const float2 t = __fmul2_rn(w, make_float2(a.x, a.x));
    return __ffma2_rn(make_float2(-w.y, w.x), make_float2(a.y, a.y), t);
}
#endif
template <typename C, typename T> __device__ __forceinline__ C cscale(C a, T s) { C r; r.x = a.x * s; r.y = a.y * s; return r; }
#ifdef __CUDA_ARCH__
__device__ __forceinline__ float2 cscale(float2 a, float s) { return __fmul2_rn(a, make_float2(s, s)); }
#endif
// multiply by s*i, s = +1 or -1 (compile time)
template <int S, typename C> __device__ __forceinline__ C cmul_i(C a) {
    C r;
    if constexpr (S > 0) { r.x = -a.y; r.y = a.x; } else { r.x = a.y; r.y = -a.x; }
    return r;
}

// ---------------------------------------------------------------------------------------------
// Compile-time cos/sin of 2*pi*num/den, evaluated by the compiler in double:
// exact octant reduction in integers, then a Taylor series on [0, pi/4].
// ---------------------------------------------------------------------------------------------
namespace ct {
constexpr double PI = 3.14159265358979323846264338327950288;

constexpr double sin_taylor(double x) {
    double term = x, sum = x, x2 = x * x;
    for (int n = 1; n < 16; ++n) { term *= -x2 / ((2 * n) * (2 * n + 1)); sum += term; }
    return sum;
}
constexpr double cos_taylor(double x) {
    double term = 1.0, sum = 1.0, x2 = x * x;
    for (int n = 1; n < 16; ++n) { term *= -x2 / ((2 * n - 1) * (2 * n)); sum += term; }
    return sum;
}
struct cs { double c, s; };
// angle = 2*pi*num/den, any integer num, den > 0
constexpr cs cossin(long long num, long long den) {
    long long n = num % den;
    if (n < 0) n += den;
    // work in units of 1/(8 den) of a turn: a = 8n, full turn = 8 den
    long long a = 8 * n, full = 8 * den, half = 4 * den, quarter = 2 * den, oct = den;
    bool neg_s = false, neg_c = false, swap = false;
    if (a > half) { a = full - a; neg_s = true; }            // cos(2pi-a)=cos a, sin = -sin
    if (a > quarter) { a = half - a; neg_c = true; }         // cos(pi-a)=-cos a, sin = sin
    if (a > oct) { a = quarter - a; swap = true; }           // cos(pi/2-a)=sin a
    double x = 2.0 * PI * (double)a / (double)full;
    double c = cos_taylor(x), s = sin_taylor(x);
    if (a == 0) { c = 1.0; s = 0.0; }
    if (swap) { double t = c; c = s; s = t; }
    if (neg_c) c = -c;
    if (neg_s) s = -s;
    return cs{c, s};
}
}  // namespace ct

// a * exp(DIR * 2 pi i NUM / DEN) with the trivial rotations done without multiplications.
template <int NUM, int DEN, int DIR, typename T, bool PACK = true>
__device__ __forceinline__ cx<T> mul_root(cx<T> a) {
    constexpr int n = ((NUM % DEN) + DEN) % DEN;
    if constexpr (n == 0) {
        return a;
    } else if constexpr (4 * n == DEN) {
        return cmul_i<DIR>(a);
    } else if constexpr (2 * n == DEN) {
        return mk<T>(-a.x, -a.y);
    } else if constexpr (4 * n == 3 * DEN) {
        return cmul_i<-DIR>(a);
    } else {
        constexpr ct::cs w = ct::cossin(n, DEN);
        constexpr T c = (T)w.c;
        constexpr T s = (T)(DIR > 0 ? w.s : -w.s);
#ifdef __CUDA_ARCH__
        if constexpr (sizeof(T) == 4 && PACK) {
            const float2 t = __fmul2_rn(a, make_float2(c, c));
            return __ffma2_rn(make_float2(-a.y, a.x), make_float2(s, s), t);
        } else
#endif
        {
            cx<T> r;
            r.x = a.x * c - a.y * s;
            r.y = a.x * s + a.y * c;
            return r;
        }
    }
}

// ---------------------------------------------------------------------------------------------
// In-register DFT of length R, natural order in and out.  Decimation in time:
//   R = R1*R2, x[R1*a + q] -> Y_q = DFT_R2, X[k + s*R2] = sum_q W_R1^{qs} (W_R^{qk} Y_q[k]).
// ---------------------------------------------------------------------------------------------
template <int R, int DIR, typename T>
__device__ __forceinline__ void dft(cx<T> (&v)[R]);

// combine step unrolled over k at compile time (the twiddle exponent q*k must be a template arg)
template <int R, int R1, int R2, int DIR, typename T, int K, int Q>
__device__ __forceinline__ void combine_tw(cx<T> (&sub)[R1][R2], cx<T> (&t)[R1]) {
    if constexpr (Q < R1) {
        t[Q] = mul_root<Q * K, R, DIR, T>(sub[Q][K]);
        combine_tw<R, R1, R2, DIR, T, K, Q + 1>(sub, t);
    }
}

template <int R, int R1, int R2, int DIR, typename T, int K>
__device__ __forceinline__ void combine(cx<T> (&sub)[R1][R2], cx<T> (&v)[R]) {
    if constexpr (K < R2) {
        cx<T> t[R1];
        combine_tw<R, R1, R2, DIR, T, K, 0>(sub, t);
        dft<R1, DIR, T>(t);
#pragma unroll
        for (int s = 0; s < R1; ++s) v[K + s * R2] = t[s];
        combine<R, R1, R2, DIR, T, K + 1>(sub, v);
    }
}

template <int R, int DIR, typename T>
__device__ __forceinline__ void dft(cx<T> (&v)[R]) {
    using C = cx<T>;
    if constexpr (R == 1) {
        return;
    } else if constexpr (R == 2) {
        C a = v[0], b = v[1];
        v[0] = cadd(a, b);
        v[1] = csub(a, b);
    } else if constexpr (R == 3) {
        constexpr T h = (T)0.86602540378443864676372317075293618;   // sqrt(3)/2
        C s = cadd(v[1], v[2]), d = csub(v[1], v[2]);
        C m = mk<T>(v[0].x - (T)0.5 * s.x, v[0].y - (T)0.5 * s.y);
        C id = cmul_i<DIR>(d);                                         // DIR * i * d
        v[0] = cadd(v[0], s);
        v[1] = mk<T>(m.x + h * id.x, m.y + h * id.y);
        v[2] = mk<T>(m.x - h * id.x, m.y - h * id.y);
    } else if constexpr (R == 4) {
        C t0 = cadd(v[0], v[2]), t1 = csub(v[0], v[2]);
        C t2 = cadd(v[1], v[3]), d = csub(v[1], v[3]);
        C id = cmul_i<DIR>(d);
        v[0] = cadd(t0, t2);
        v[2] = csub(t0, t2);
        v[1] = cadd(t1, id);
        v[3] = csub(t1, id);
    } else if constexpr (R == 5) {
        // X_k = x0 + sum_{j=1..4} x_j w^(jk), w = exp(DIR 2 pi i/5): with s1 = x1+x4, s2 = x2+x3, d1 = x1-x4, d2 = x2-x3,
        // X_{1,4} = x0 + c1 s1 + c2 s2 +- DIR i (k1 d1 + k2 d2),  X_{2,3} = x0 + c2 s1 + c1 s2 +- DIR i (k2 d1 - k1 d2)
        constexpr T c1 = (T)0.30901699437494742410229341718281906;    // cos(2 pi/5)
        constexpr T c2 = (T)-0.80901699437494742410229341718281906;   // cos(4 pi/5)
        constexpr T k1 = (T)0.95105651629515357211643933337938214;    // sin(2 pi/5)
        constexpr T k2 = (T)0.58778525229247312916870595463907277;    // sin(4 pi/5)
        const C s1 = cadd(v[1], v[4]), s2 = cadd(v[2], v[3]), d1 = csub(v[1], v[4]), d2 = csub(v[2], v[3]);
        const C a1 = mk<T>(v[0].x + c1 * s1.x + c2 * s2.x, v[0].y + c1 * s1.y + c2 * s2.y);
        const C a2 = mk<T>(v[0].x + c2 * s1.x + c1 * s2.x, v[0].y + c2 * s1.y + c1 * s2.y);
        const C b1 = cmul_i<DIR>(mk<T>(k1 * d1.x + k2 * d2.x, k1 * d1.y + k2 * d2.y));
        const C b2 = cmul_i<DIR>(mk<T>(k2 * d1.x - k1 * d2.x, k2 * d1.y - k1 * d2.y));
        v[0] = mk<T>(v[0].x + s1.x + s2.x, v[0].y + s1.y + s2.y);
        v[1] = cadd(a1, b1);
        v[4] = csub(a1, b1);
        v[2] = cadd(a2, b2);
        v[3] = csub(a2, b2);
    } else if constexpr (R == 7) {
        // X_k = x0 + sum_{j=1..3} [ s_j cos(2 pi jk/7) + DIR i d_j sin(2 pi jk/7) ],  s_j = x_j + x_{7-j}, d_j = x_j - x_{7-j};
        // X_{7-k} is the same with the sign of the second term flipped
        constexpr T c1 = (T)0.62348980185873353052500488400423981;    // cos(2 pi/7)
        constexpr T c2 = (T)-0.22252093395631440428890256449679476;   // cos(4 pi/7)
        constexpr T c3 = (T)-0.90096886790241912623610231950744505;   // cos(6 pi/7)
        constexpr T k1 = (T)0.78183148246802980870844452667405775;    // sin(2 pi/7)
        constexpr T k2 = (T)0.97492791218182360701813168299393122;    // sin(4 pi/7)
        constexpr T k3 = (T)0.43388373911755812047576833284835875;    // sin(6 pi/7)
        const C s1 = cadd(v[1], v[6]), s2 = cadd(v[2], v[5]), s3 = cadd(v[3], v[4]);
        const C d1 = csub(v[1], v[6]), d2 = csub(v[2], v[5]), d3 = csub(v[3], v[4]);
        const C a1 = mk<T>(v[0].x + c1 * s1.x + c2 * s2.x + c3 * s3.x, v[0].y + c1 * s1.y + c2 * s2.y + c3 * s3.y);
        const C a2 = mk<T>(v[0].x + c2 * s1.x + c3 * s2.x + c1 * s3.x, v[0].y + c2 * s1.y + c3 * s2.y + c1 * s3.y);
        const C a3 = mk<T>(v[0].x + c3 * s1.x + c1 * s2.x + c2 * s3.x, v[0].y + c3 * s1.y + c1 * s2.y + c2 * s3.y);
        const C b1 = cmul_i<DIR>(mk<T>(k1 * d1.x + k2 * d2.x + k3 * d3.x, k1 * d1.y + k2 * d2.y + k3 * d3.y));
        const C b2 = cmul_i<DIR>(mk<T>(k2 * d1.x - k3 * d2.x - k1 * d3.x, k2 * d1.y - k3 * d2.y - k1 * d3.y));
        const C b3 = cmul_i<DIR>(mk<T>(k3 * d1.x - k1 * d2.x + k2 * d3.x, k3 * d1.y - k1 * d2.y + k2 * d3.y));
        v[0] = mk<T>(v[0].x + s1.x + s2.x + s3.x, v[0].y + s1.y + s2.y + s3.y);
        v[1] = cadd(a1, b1);
        v[6] = csub(a1, b1);
        v[2] = cadd(a2, b2);
        v[5] = csub(a2, b2);
        v[3] = cadd(a3, b3);
        v[4] = csub(a3, b3);
    } else {
        constexpr int R1 = (R % 4 == 0) ? 4 : ((R % 2 == 0) ? 2 : ((R % 3 == 0) ? 3 : ((R % 5 == 0) ? 5 : 7)));
        constexpr int R2 = R / R1;
        static_assert(R1 * R2 == R, "radix must be 2^a 3^b 5^c 7^d");
        C sub[R1][R2];
#pragma unroll
        for (int q = 0; q < R1; ++q)
#pragma unroll
            for (int a = 0; a < R2; ++a) sub[q][a] = v[R1 * a + q];
#pragma unroll
        for (int q = 0; q < R1; ++q) dft<R2, DIR, T>(sub[q]);
        combine<R, R1, R2, DIR, T, 0>(sub, v);
    }
}

}  // namespace fft3d
