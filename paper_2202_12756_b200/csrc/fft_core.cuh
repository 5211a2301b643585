// fft_core.cuh -- a length-N complex FFT spread over N/P threads, P points per thread in
// registers, radix-R[s] stages joined by shared-memory exchanges (Stockham autosort, natural
// order in and out).
//
// Thread t of an FFT holds elements e = t + m*S (S = N/P, m = 0..P-1) in v[m] -- both on entry
// (input order) and on exit (output order).  Stage s (radix r, Ns = product of earlier radices)
// runs P/r butterflies per thread; butterfly u takes v[u + i*P/r], i < r, i.e. elements
// j + i*N/r with j = t + u*S, multiplies by exp(DIR 2 pi i * i*k/(Ns r)), k = j mod Ns, applies
// DFT_r and scatters to elements (j/Ns)*Ns*r + k + i*Ns.  For the last stage that scatter lands
// on the thread's own elements again, so the result stays in registers.
//
// Shared-memory addressing is kept LINEAR in (thread part) + (compile-time part): every LDS/STS
// of the unrolled stages is `per-thread base register + immediate`, so the exchanges cost no
// integer instructions beyond a handful of bases per stage.
#pragma once
#include "fft_radix.cuh"

namespace fft3d {

template <int N_, int P_, int R0, int R1 = 1, int R2 = 1, int R3 = 1, int R4 = 1>
struct FftCfg {
    static constexpr int N = N_, P = P_, S = N_ / P_;
    static constexpr int NST = 1 + (R1 > 1) + (R2 > 1) + (R3 > 1) + (R4 > 1);
    __host__ __device__ static constexpr int radix(int s) {
        return s == 0 ? R0 : s == 1 ? R1 : s == 2 ? R2 : s == 3 ? R3 : R4;
    }
    __host__ __device__ static constexpr int ns(int s) {          // product of radices before stage s
        int p = 1;
        for (int i = 0; i < s; ++i) p *= radix(i);
        return p;
    }
    __host__ __device__ static constexpr int twoff(int s) {       // table offset of stage s (s >= 1)
        int o = 0;
        for (int i = 1; i < s; ++i) o += (radix(i) - 1) * ns(i);
        return o;
    }
    static constexpr int TWN = twoff(NST);                        // total twiddle entries
    static_assert(R0 * R1 * R2 * R3 * R4 == N_, "radices must multiply to N");
    static_assert(N_ % P_ == 0, "P must divide N");
    static_assert(P_ % R0 == 0 && P_ % R1 == 0 && P_ % R2 == 0 && P_ % R3 == 0 && P_ % R4 == 0,
                  "every radix must divide P");
};

// Shared-memory slot of element e of one FFT: (e + e/PADR) * TC + c.
//   TC   = elements between consecutive e (the tile width of a strided pass; 1 for a row pass)
//   PADR = one element (row) of padding after every PADR elements, 0 = none: breaks the
//          power-of-two stride of the first exchange (bank conflicts)
//   c    = per-thread constant (tile column, or the start of the thread's row)
template <int TC_, int PADR_>
struct SmLayout {
    static constexpr int TC = TC_, PADR = PADR_;
    int c;
    __device__ __forceinline__ int at(int e) const {
        if constexpr (PADR_ > 0) return (e + e / PADR_) * TC_ + c;
        else return e * TC_ + c;
    }
    // slot offset contributed by a compile-time element offset (valid when the split is additive)
    __host__ __device__ static constexpr int off(int econst) {
        return (PADR_ > 0 ? econst + econst / PADR_ : econst) * TC_;
    }
};

struct CtaSync {
    __device__ __forceinline__ void operator()() const { __syncthreads(); }
};
// named barrier over the first `NT` threads of the CTA (warp-specialised kernels)
template <int ID, int NT>
struct NamedSync {
    __device__ __forceinline__ void operator()() const {
        asm volatile("bar.sync %0, %1;" ::"n"(ID), "n"(NT) : "memory");
    }
};

template <class Cfg, class Lay>
struct StageAddr {
    static constexpr int S = Cfg::S;
    // the (thread part) + (compile-time part) split of slot addresses is exact when no carry can
    // cross a padding boundary
    // (S a multiple of the padding period; or, for two-stage transforms -- whose only scatter is
    // stage 0 -- S a divisor of it: then (t + m*S)/PADR = (m*S)/PADR for every t < S)
    static constexpr bool LINEAR = (Lay::PADR == 0) ||
        (Lay::PADR == Cfg::radix(0) && (S % Lay::PADR == 0 || (Lay::PADR % S == 0 && Cfg::NST == 2)));
};

// Read the thread's P elements (t + m*S) from shared memory.
template <class Cfg, typename T, class Lay>
__device__ __forceinline__ void read_own(cx<T> (&v)[Cfg::P], const cx<T>* __restrict__ sm, int t, const Lay& lay) {
    constexpr int P = Cfg::P, S = Cfg::S;
    if constexpr (StageAddr<Cfg, Lay>::LINEAR) {
        const cx<T>* b = sm + lay.at(t);
#pragma unroll
        for (int m = 0; m < P; ++m) v[m] = b[Lay::off(m * S)];
    } else {
#pragma unroll
        for (int m = 0; m < P; ++m) v[m] = sm[lay.at(t + m * S)];
    }
}

template <class Cfg, typename T, class Lay>
__device__ __forceinline__ void write_own(const cx<T> (&v)[Cfg::P], cx<T>* __restrict__ sm, int t, const Lay& lay) {
    constexpr int P = Cfg::P, S = Cfg::S;
    if constexpr (StageAddr<Cfg, Lay>::LINEAR) {
        cx<T>* b = sm + lay.at(t);
#pragma unroll
        for (int m = 0; m < P; ++m) b[Lay::off(m * S)] = v[m];
    } else {
#pragma unroll
        for (int m = 0; m < P; ++m) sm[lay.at(t + m * S)] = v[m];
    }
}

struct NoHook {
    __device__ __forceinline__ void operator()() const {}
};

// One stage (and, recursively, the following ones).  `before_scatter` runs once, after the first butterfly of
// stage 0 has been computed in registers and before anything is written to `sm` (transforms with more than one
// stage only): kernels whose exchange buffer may still be busy wait for it there, behind the arithmetic.
template <class Cfg, int SI, int DIR, typename T, class Lay, class Sync, class Hook = NoHook>
__device__ __forceinline__ void fft_stages(cx<T> (&v)[Cfg::P], cx<T>* __restrict__ sm,
                                           const cx<T>* __restrict__ tw, int t, const Lay& lay,
                                           const Sync& sync, const Hook& before_scatter = Hook{}) {
    using C = cx<T>;
    constexpr int r = Cfg::radix(SI), Ns = Cfg::ns(SI), P = Cfg::P, S = Cfg::S, B = P / r;
    constexpr bool last = (SI == Cfg::NST - 1);
    constexpr bool LIN = StageAddr<Cfg, Lay>::LINEAR;
    // how j = t + u*S splits into (j / Ns, j % Ns)
    constexpr bool CASE_A = (S % Ns == 0);                 // j%Ns = t%Ns, j/Ns = t/Ns + u*S/Ns
    constexpr bool CASE_B = !CASE_A && (Ns % S == 0);      // j%Ns = t + (u%(Ns/S))*S, j/Ns = u/(Ns/S)
    if constexpr (!last && SI > 0) sync();                 // everyone has read the previous exchange

    int jr_run = 0, erun = 0;                              // thread parts of j%Ns and of the scatter base
    if constexpr (CASE_A) { jr_run = t % Ns; erun = (t / Ns) * (Ns * r) + jr_run; }
    else if constexpr (CASE_B) { jr_run = t; erun = t; }
    const C* twb = tw + Cfg::twoff(SI) + jr_run;
    C* wb = sm + ((LIN && (CASE_A || CASE_B)) ? lay.at(erun) : 0);

#pragma unroll
    for (int u = 0; u < B; ++u) {
        C a[r];
#pragma unroll
        for (int i = 0; i < r; ++i) a[i] = v[u + i * B];
        // compile-time parts
        int jr_c = 0, e_c = 0;
        if constexpr (CASE_A) { jr_c = 0; e_c = u * (S / Ns) * (Ns * r); }
        else if constexpr (CASE_B) { jr_c = (u % (Ns / S)) * S; e_c = (u / (Ns / S)) * (Ns * r) + jr_c; }
        if constexpr (Ns > 1) {
            if constexpr (CASE_A || CASE_B) {
#pragma unroll
                for (int i = 1; i < r; ++i) a[i] = cmul(a[i], twb[jr_c + (i - 1) * Ns]);
            } else {
                const int k = (t + u * S) % Ns;
                const C* twk = tw + Cfg::twoff(SI) + k;
#pragma unroll
                for (int i = 1; i < r; ++i) a[i] = cmul(a[i], twk[(i - 1) * Ns]);
            }
        }
        dft<r, DIR, T>(a);
        if constexpr (SI == 0 && !last) {
            if (u == 0) before_scatter();
        }
        if constexpr (last) {
#pragma unroll
            for (int i = 0; i < r; ++i) v[u + i * B] = a[i];
        } else if constexpr (LIN && (CASE_A || CASE_B)) {
#pragma unroll
            for (int i = 0; i < r; ++i) wb[Lay::off(e_c + i * Ns)] = a[i];
        } else {
            const int j = t + u * S;
            const int j0 = (j / Ns) * (Ns * r) + (j % Ns);
#pragma unroll
            for (int i = 0; i < r; ++i) sm[lay.at(j0 + i * Ns)] = a[i];
        }
    }
    if constexpr (!last) {
        sync();
        read_own<Cfg, T, Lay>(v, sm, t, lay);
        fft_stages<Cfg, SI + 1, DIR, T, Lay, Sync>(v, sm, tw, t, lay, sync);
    }
}

// Copy the plan's forward twiddle table (exp(-2 pi i ...)) into shared memory, conjugated for
// the inverse direction.
template <int DIR, typename T>
__device__ __forceinline__ void load_twiddles(cx<T>* dst, const cx<T>* __restrict__ src, int n,
                                              int tid, int nthreads) {
    for (int i = tid; i < n; i += nthreads) {
        cx<T> w = src[i];
        if constexpr (DIR > 0) w.y = -w.y;
        dst[i] = w;
    }
}

}  // namespace fft3d
