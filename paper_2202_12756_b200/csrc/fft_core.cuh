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

// One stage (and, recursively, the following ones).  `Idx` maps an element index of this FFT
// to a shared-memory slot (tile column / row padding folded in).  `sync` is a CTA barrier.
template <class Cfg, int SI, int DIR, typename T, class Idx>
__device__ __forceinline__ void fft_stages(cx<T> (&v)[Cfg::P], cx<T>* __restrict__ sm,
                                           const cx<T>* __restrict__ tw, int t, const Idx& idx) {
    using C = cx<T>;
    constexpr int r = Cfg::radix(SI), Ns = Cfg::ns(SI), P = Cfg::P, S = Cfg::S, B = P / r;
    constexpr bool last = (SI == Cfg::NST - 1);
    if constexpr (!last && SI > 0) __syncthreads();      // everyone has read the previous exchange
#pragma unroll
    for (int u = 0; u < B; ++u) {
        C a[r];
#pragma unroll
        for (int i = 0; i < r; ++i) a[i] = v[u + i * B];
        const int j = t + u * S;
        if constexpr (Ns > 1) {
            const int k = j % Ns;
            const C* twk = tw + Cfg::twoff(SI) + k;
#pragma unroll
            for (int i = 1; i < r; ++i) a[i] = cmul(a[i], twk[(i - 1) * Ns]);
        }
        dft<r, DIR, T>(a);
        if constexpr (last) {
#pragma unroll
            for (int i = 0; i < r; ++i) v[u + i * B] = a[i];
        } else {
            const int j0 = (j / Ns) * (Ns * r) + (j % Ns);
#pragma unroll
            for (int i = 0; i < r; ++i) sm[idx(j0 + i * Ns)] = a[i];
        }
    }
    if constexpr (!last) {
        __syncthreads();
#pragma unroll
        for (int m = 0; m < P; ++m) v[m] = sm[idx(t + m * S)];
        fft_stages<Cfg, SI + 1, DIR, T, Idx>(v, sm, tw, t, idx);
    }
}

// Copy the plan's forward twiddle table (exp(-2 pi i ...)) into shared memory, conjugated for
// the inverse direction.
template <int DIR, typename T>
__device__ __forceinline__ void load_twiddles(cx<T>* dst, const cx<T>* __restrict__ src, int n) {
    for (int i = threadIdx.x; i < n; i += blockDim.x) {
        cx<T> w = src[i];
        if constexpr (DIR > 0) w.y = -w.y;
        dst[i] = w;
    }
}

}  // namespace fft3d
