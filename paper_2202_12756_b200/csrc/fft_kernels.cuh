// fft_kernels.cuh -- the three kinds of full-array passes of the slab 3D FFT:
//
//   fft_z_r2c_kernel   pass F1: rows of Nz reals -> Nz/2 packed complex (paper step 1, z half)
//   fft_z_c2r_kernel   pass I3: the mirror image, with the 1/(NxNyNz) normalisation fused
//   fft_strided_kernel passes F2, F3, I1, I2: C2C FFT down a strided axis on a [N rows][TC cols]
//                      tile; the row index may be split as row = q*L + l on the input or the
//                      output side, which is how the paper's local transpose + all-to-all + chunk
//                      transpose (steps 2-4) are folded into the y pass as pure addressing.
//
// "Packed" complex rows: the z pass keeps Nz/2 columns; column 0 holds (X[0], X[Nz/2]) -- both
// real after an R2C -- as one complex number.  The strided passes are linear, so column 0 then
// carries A + iB with A, B the transforms of two real planes; fft3d_fixup.cu separates them.
#pragma once
#include "fft_core.cuh"

namespace fft3d {

struct StridedArgs {
    const void* in;
    void* out;
    const void* col0;            // if non-null: column 0 of the input is read from here instead
    const void* tw;              // forward stage twiddles (device), Cfg::TWN entries
    long long ntiles;            // = n_a * ntz
    int ntz;                     // column tiles per row
    int ncols;                   // valid columns
    int a_lo;                    // tile id -> a = id / ntz -> (a / a_lo, a % a_lo)
    int L;                       // rows per virtual slab (row = q*L + l) for the *_SLAB side
    long long in_hi, in_lo;      // element offset of tile (a_hi, a_lo): a_hi*in_hi + a_lo*in_lo
    long long out_hi, out_lo;
    long long c0_hi, c0_lo;
    long long in_rq, in_rl;      // element offset of row (q, l): q*in_rq + l*in_rl  (q = 0 if !IN_SLAB)
    long long out_rq, out_rl;
    long long c0_rl;
};

struct ZArgs {
    const void* in;
    void* out;
    const void* tw;              // stage twiddles for the M = Nz/2 point FFT
    const void* twz;             // exp(-2 pi i k / Nz), k < M
    long long nrows;
    double scale;                // C2R only: 1/(Nx Ny Nz)
};

// row padding of shared-memory tiles: one extra row every PADR rows (0 = none)
template <class Cfg, int ROW_BYTES>
struct TilePad {
    static constexpr int r0 = Cfg::radix(0);
    static constexpr int PADR = (ROW_BYTES < 128 && Cfg::NST > 1 && r0 % 4 == 0) ? r0 : 0;
    static constexpr int ROWS = Cfg::N + (PADR ? Cfg::N / PADR : 0);
};

template <int PADR, int TC>
struct TileIdx {
    int c;
    __device__ __forceinline__ int operator()(int e) const {
        if constexpr (PADR > 0) return (e + e / PADR) * TC + c;
        else return e * TC + c;
    }
};

template <bool SLAB>
__device__ __forceinline__ long long row_offset(int row, int L, float invL, long long rq, long long rl) {
    if constexpr (SLAB) {
        int q = __float2int_rz(((float)row + 0.5f) * invL);   // row < 2^22: exact floor(row/L)
        int l = row - q * L;
        return (long long)q * rq + (long long)l * rl;
    } else {
        return (long long)row * rl;
    }
}

template <class Cfg, int TC, int DIR, bool IN_SLAB, bool OUT_SLAB, typename T, int MINB>
__global__ void __launch_bounds__(Cfg::S * TC, MINB) fft_strided_kernel(const StridedArgs a) {
    using C = cx<T>;
    constexpr int P = Cfg::P, S = Cfg::S;
    using Pad = TilePad<Cfg, TC * (int)sizeof(C)>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C* tw = reinterpret_cast<C*>(smem_raw);
    C* tile = tw + ((Cfg::TWN + 1) & ~1);
    load_twiddles<DIR, T>(tw, reinterpret_cast<const C*>(a.tw), Cfg::TWN);

    const int c = threadIdx.x % TC, t = threadIdx.x / TC;
    const TileIdx<Pad::PADR, TC> idx{c};
    const float invL = 1.0f / (float)a.L;

    for (long long tid = blockIdx.x; tid < a.ntiles; tid += gridDim.x) {
        const int tz = (int)(tid % a.ntz);
        const long long aa = tid / a.ntz;
        const long long a_hi = aa / a.a_lo, a_l = aa % a.a_lo;
        const int col = tz * TC + c;
        const bool ok = col < a.ncols;
        const C* in = reinterpret_cast<const C*>(a.in) + (a_hi * a.in_hi + a_l * a.in_lo + col);
        C* out = reinterpret_cast<C*>(a.out) + (a_hi * a.out_hi + a_l * a.out_lo + col);
        long long in_rl = a.in_rl;
        if (a.col0 != nullptr && col == 0) {      // packed column 0 comes from the side buffer
            in = reinterpret_cast<const C*>(a.col0) + (a_hi * a.c0_hi + a_l * a.c0_lo);
            in_rl = a.c0_rl;
        }
        C v[P];
#pragma unroll
        for (int m = 0; m < P; ++m) {
            const long long off = row_offset<IN_SLAB>(t + m * S, a.L, invL, a.in_rq, in_rl);
            v[m] = ok ? in[off] : mk<T>((T)0, (T)0);
        }
        if constexpr (Cfg::NST > 1) __syncthreads();   // twiddles loaded / previous tile fully read
        fft_stages<Cfg, 0, DIR, T>(v, tile, tw, t, idx);
        if (ok) {
#pragma unroll
            for (int m = 0; m < P; ++m) {
                const long long off = row_offset<OUT_SLAB>(t + m * S, a.L, invL, a.out_rq, a.out_rl);
                out[off] = v[m];
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// z passes.  Cfg::N = M = Nz/2.  RPB rows per CTA iteration, S = M/P threads per row.
// ---------------------------------------------------------------------------------------------
template <class Cfg>
struct RowPad {
    static constexpr int r0 = Cfg::radix(0);
    static constexpr int PADR = r0;                                   // pad one element every r0
    static constexpr int PITCH = Cfg::N + Cfg::N / PADR + 1;
};

template <int PADR>
struct RowIdx {
    int base;
    __device__ __forceinline__ int operator()(int e) const { return base + e + e / PADR; }
};

template <class Cfg, int RPB, typename T, int MINB>
__global__ void __launch_bounds__(Cfg::S * RPB, MINB) fft_z_r2c_kernel(const ZArgs a) {
    using C = cx<T>;
    constexpr int P = Cfg::P, S = Cfg::S, M = Cfg::N;
    using Pad = RowPad<Cfg>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C* tw = reinterpret_cast<C*>(smem_raw);
    C* twz = tw + ((Cfg::TWN + 1) & ~1);
    C* rows = twz + M;
    load_twiddles<-1, T>(tw, reinterpret_cast<const C*>(a.tw), Cfg::TWN);
    load_twiddles<-1, T>(twz, reinterpret_cast<const C*>(a.twz), M);

    const int t = threadIdx.x % S, rr = threadIdx.x / S;
    const RowIdx<Pad::PADR> idx{rr * Pad::PITCH};
    const long long ngroups = (a.nrows + RPB - 1) / RPB;

    for (long long g = blockIdx.x; g < ngroups; g += gridDim.x) {
        const long long row = g * RPB + rr;
        const bool ok = row < a.nrows;
        // a row of Nz reals read as M (even, odd) pairs: z[m] = x[2m] + i x[2m+1]
        const C* in = reinterpret_cast<const C*>(a.in) + row * M;
        C* out = reinterpret_cast<C*>(a.out) + row * M;
        C v[P];
#pragma unroll
        for (int m = 0; m < P; ++m) v[m] = ok ? in[t + m * S] : mk<T>((T)0, (T)0);
        __syncthreads();                               // tables loaded / previous group fully read
        fft_stages<Cfg, 0, -1, T>(v, rows, tw, t, idx);
        if constexpr (Cfg::NST > 1) __syncthreads();
#pragma unroll
        for (int m = 0; m < P; ++m) rows[idx(t + m * S)] = v[m];
        __syncthreads();
        // X[k] = (Z[k] + conj Z[M-k])/2 - (i/2) w^k (Z[k] - conj Z[M-k]),  w = exp(-2 pi i/Nz)
#pragma unroll
        for (int m = 0; m < P; ++m) {
            const int k = t + m * S;
            C r;
            if (k == 0) {
                r = mk<T>(v[m].x + v[m].y, v[m].x - v[m].y);          // (X[0], X[Nz/2]) packed
            } else {
                const C zm = cconj(rows[idx(M - k)]);
                const C e = cadd(v[m], zm), d = csub(v[m], zm);
                const C w = cmul(twz[k], d);
                r = mk<T>((T)0.5 * (e.x + w.y), (T)0.5 * (e.y - w.x));
            }
            if (ok) out[k] = r;
        }
    }
}

template <class Cfg, int RPB, typename T, int MINB>
__global__ void __launch_bounds__(Cfg::S * RPB, MINB) fft_z_c2r_kernel(const ZArgs a) {
    using C = cx<T>;
    constexpr int P = Cfg::P, S = Cfg::S, M = Cfg::N;
    using Pad = RowPad<Cfg>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C* tw = reinterpret_cast<C*>(smem_raw);
    C* twz = tw + ((Cfg::TWN + 1) & ~1);
    C* rows = twz + M;
    load_twiddles<+1, T>(tw, reinterpret_cast<const C*>(a.tw), Cfg::TWN);
    load_twiddles<+1, T>(twz, reinterpret_cast<const C*>(a.twz), M);     // conj: exp(+2 pi i k/Nz)

    const int t = threadIdx.x % S, rr = threadIdx.x / S;
    const RowIdx<Pad::PADR> idx{rr * Pad::PITCH};
    const long long ngroups = (a.nrows + RPB - 1) / RPB;
    const T scale = (T)a.scale;

    for (long long g = blockIdx.x; g < ngroups; g += gridDim.x) {
        const long long row = g * RPB + rr;
        const bool ok = row < a.nrows;
        const C* in = reinterpret_cast<const C*>(a.in) + row * M;
        C* out = reinterpret_cast<C*>(a.out) + row * M;
        C v[P];
#pragma unroll
        for (int m = 0; m < P; ++m) v[m] = ok ? in[t + m * S] : mk<T>((T)0, (T)0);
        __syncthreads();                               // tables loaded / previous group fully read
#pragma unroll
        for (int m = 0; m < P; ++m) rows[idx(t + m * S)] = v[m];
        __syncthreads();
        // Z[k] = (X[k] + conj X[M-k]) + i conj(w)^k (X[k] - conj X[M-k]); column 0 holds the real
        // pair (X[0], X[Nz/2]): Z[0] = (X0 + XM) + i (X0 - XM).
#pragma unroll
        for (int m = 0; m < P; ++m) {
            const int k = t + m * S;
            if (k == 0) {
                v[m] = mk<T>(v[m].x + v[m].y, v[m].x - v[m].y);
            } else {
                const C xm = cconj(rows[idx(M - k)]);
                const C e = cadd(v[m], xm), d = csub(v[m], xm);
                const C w = cmul(twz[k], d);
                v[m] = mk<T>(e.x - w.y, e.y + w.x);
            }
        }
        if constexpr (Cfg::NST > 1) __syncthreads();
        fft_stages<Cfg, 0, +1, T>(v, rows, tw, t, idx);
        // z[m] = x[2m] + i x[2m+1]; scale by 1/(Nx Ny Nz)
        if (ok) {
#pragma unroll
            for (int m = 0; m < P; ++m) out[t + m * S] = mk<T>(v[m].x * scale, v[m].y * scale);
        }
    }
}

}  // namespace fft3d
