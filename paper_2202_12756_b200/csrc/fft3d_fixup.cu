// fft3d_fixup.cu -- the two plane-sized kernels that go with the packed column 0 of the
// intermediate arrays.
//
// After the z-axis R2C, X[0] and X[Nz/2] of every row are real, so the passes keep Nz/2 columns
// and store (X[0], X[Nz/2]) as one complex number in column 0.  The y and x transforms are
// linear, so at the end column 0 holds C = A + iB, where A and B are the 2D transforms of two
// REAL planes and therefore Hermitian: A(k) = (C(k) + conj C(-k))/2, B(k) = (C(k) - conj C(-k))/(2i),
// k = (kx, ky) mod (Nx, Ny).  unpack_nyquist separates them into the planes kz = 0 and kz = Nz/2
// of the output (Eq. (3)/(4)).  pack_nyquist is the inverse step; it first takes
// the Hermitian part of each plane, which is all that Eq. (2)+(3) lets through (reading R8).
#include <cuda_runtime.h>

#include "fft_radix.cuh"

namespace fft3d {

struct PlaneArgs {
    const void* src;
    void* dst;
    int Nx, Ny, L, M;
};

// grid cap of the plane-sized grid-stride kernels below: 16 blocks of 256 threads per SM of the current device
static long long grid_cap() {
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms < 1) {
        cudaGetLastError();
        sms = 148;                                    // B200
    }
    return (long long)sms * 16;
}

__device__ __forceinline__ long long slab_row(int kx, int ky, int Nx, int L) {
    const int q = ky / L, l = ky - q * L;
    return ((long long)q * Nx + kx) * L + l;
}

template <typename T>
__global__ void unpack_nyquist_kernel(const PlaneArgs a) {
    using C = cx<T>;
    const long long n = (long long)a.Nx * a.Ny;
    const long long pitch = a.M + 1;
    C* out = reinterpret_cast<C*>(a.dst);
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n;
         i += (long long)gridDim.x * blockDim.x) {
        const int kx = (int)(i / a.Ny), ky = (int)(i % a.Ny);
        const int mx = kx == 0 ? 0 : a.Nx - kx, my = ky == 0 ? 0 : a.Ny - ky;
        const long long j = (long long)mx * a.Ny + my;
        if (j < i) continue;                      // the pair is handled by its lower index
        const long long r1 = slab_row(kx, ky, a.Nx, a.L) * pitch;
        const long long r2 = slab_row(mx, my, a.Nx, a.L) * pitch;
        const C c1 = out[r1], c2 = out[r2];
        const C A = mk<T>((T)0.5 * (c1.x + c2.x), (T)0.5 * (c1.y - c2.y));
        const C B = mk<T>((T)0.5 * (c1.y + c2.y), (T)-0.5 * (c1.x - c2.x));
        out[r1] = A;
        out[r1 + a.M] = B;
        if (j != i) {
            out[r2] = cconj(A);
            out[r2 + a.M] = cconj(B);
        }
    }
}

template <typename T>
__global__ void pack_nyquist_kernel(const PlaneArgs a) {
    using C = cx<T>;
    const long long n = (long long)a.Nx * a.Ny;
    const long long pitch = a.M + 1;
    const C* in = reinterpret_cast<const C*>(a.src);
    C* side = reinterpret_cast<C*>(a.dst);
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n;
         i += (long long)gridDim.x * blockDim.x) {
        const int kx = (int)(i / a.Ny), ky = (int)(i % a.Ny);
        const int mx = kx == 0 ? 0 : a.Nx - kx, my = ky == 0 ? 0 : a.Ny - ky;
        const long long s1 = slab_row(kx, ky, a.Nx, a.L), s2 = slab_row(mx, my, a.Nx, a.L);
        const C a1 = in[s1 * pitch], a2 = in[s2 * pitch];
        const C b1 = in[s1 * pitch + a.M], b2 = in[s2 * pitch + a.M];
        // Hermitian parts: As = (A(k) + conj A(-k))/2, Bs likewise;  side = As + i Bs
        const C As = mk<T>((T)0.5 * (a1.x + a2.x), (T)0.5 * (a1.y - a2.y));
        const C Bs = mk<T>((T)0.5 * (b1.x + b2.x), (T)0.5 * (b1.y - b2.y));
        side[s1] = mk<T>(As.x - Bs.y, As.y + Bs.x);
    }
}

// ---- distributed plans (fft3d_dist_*): the packed-column bookkeeping when the spectrum is split over G ranks ----
// Rank q owns rows ky in [q*L, (q+1)*L) of the spectrum, stored [Nx][L][M+1].  The partner C(-kx,-ky) of an own
// entry lives on rank (-ky mod Ny)/L, so the ranks first publish the planes involved as dense [Nx][L] arrays
// (extract_planes), exchange them (all-gather, or peer pointers over NVLink), and then every rank fixes up its own
// rows reading the partners from those read-only copies: no rank writes another rank's memory, nothing races.
struct DistPlaneArgs {
    const void* spec;            // own part of the spectrum [Nx][L][M+1]              (extract: source)
    void* spec_out;              // own part of the spectrum                              (unpack: destination)
    void* own;                   // own plane part [ncols][Nx][L]                         (extract: destination)
    const void* parts[16];       // every rank's plane part [ncols][Nx][L], own included  (unpack / pack: sources)
    void* side;                  // pack: own packed side buffer [Nx][L]
    int Nx, Ny, L, M, q, ncols;
};

// own[c][kx][l] = spec[kx][l][c ? M : 0]
template <typename T>
__global__ void extract_planes_kernel(const DistPlaneArgs a) {
    using C = cx<T>;
    const long long n = (long long)a.Nx * a.L;
    const C* in = reinterpret_cast<const C*>(a.spec);
    C* out = reinterpret_cast<C*>(a.own);
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n * a.ncols;
         i += (long long)gridDim.x * blockDim.x) {
        const int c = (int)(i / n);
        const long long r = i - (long long)c * n;
        out[i] = in[r * (a.M + 1) + (c ? a.M : 0)];
    }
}

// A(k) = (C(k) + conj C(-k))/2 -> column 0, B(k) = (C(k) - conj C(-k))/(2i) -> column M of the own rows
template <typename T>
__global__ void dist_unpack_kernel(const DistPlaneArgs a) {
    using C = cx<T>;
    const long long n = (long long)a.Nx * a.L;
    C* out = reinterpret_cast<C*>(a.spec_out);
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const int kx = (int)(i / a.L), l = (int)(i % a.L), ky = a.q * a.L + l;
        const int mx = kx == 0 ? 0 : a.Nx - kx, my = ky == 0 ? 0 : a.Ny - ky;
        const int mq = my / a.L, ml = my - mq * a.L;
        const C c1 = reinterpret_cast<const C*>(a.parts[a.q])[i];
        const C c2 = reinterpret_cast<const C*>(a.parts[mq])[(long long)mx * a.L + ml];
        out[i * (a.M + 1)] = mk<T>((T)0.5 * (c1.x + c2.x), (T)0.5 * (c1.y - c2.y));
        out[i * (a.M + 1) + a.M] = mk<T>((T)0.5 * (c1.y + c2.y), (T)-0.5 * (c1.x - c2.x));
    }
}

// side(k) = As(k) + i Bs(k), As / Bs the Hermitian parts of the planes kz = 0 / kz = Nz/2 (reading R8)
template <typename T>
__global__ void dist_pack_kernel(const DistPlaneArgs a) {
    using C = cx<T>;
    const long long n = (long long)a.Nx * a.L;
    C* side = reinterpret_cast<C*>(a.side);
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const int kx = (int)(i / a.L), l = (int)(i % a.L), ky = a.q * a.L + l;
        const int mx = kx == 0 ? 0 : a.Nx - kx, my = ky == 0 ? 0 : a.Ny - ky;
        const int mq = my / a.L, ml = my - mq * a.L;
        const long long j = (long long)mx * a.L + ml;
        const C* own = reinterpret_cast<const C*>(a.parts[a.q]);
        const C* oth = reinterpret_cast<const C*>(a.parts[mq]);
        const C a1 = own[i], b1 = own[n + i], a2 = oth[j], b2 = oth[n + j];
        const C As = mk<T>((T)0.5 * (a1.x + a2.x), (T)0.5 * (a1.y - a2.y));
        const C Bs = mk<T>((T)0.5 * (b1.x + b2.x), (T)0.5 * (b1.y - b2.y));
        side[i] = mk<T>(As.x - Bs.y, As.y + Bs.x);
    }
}

template <typename T>
static cudaError_t run_dist(void (*k)(const DistPlaneArgs), const DistPlaneArgs& a, cudaStream_t st) {
    const long long n = (long long)a.Nx * a.L * (a.ncols > 0 ? a.ncols : 1);
    long long blocks = (n + 255) / 256;
    if (blocks > grid_cap()) blocks = grid_cap();
    k<<<(unsigned)blocks, 256, 0, st>>>(a);
    return cudaGetLastError();
}

cudaError_t launch_dist_extract(int dtype, const DistPlaneArgs& a, cudaStream_t st) {
    return dtype == 0 ? run_dist<float>(extract_planes_kernel<float>, a, st) : run_dist<double>(extract_planes_kernel<double>, a, st);
}
cudaError_t launch_dist_unpack(int dtype, const DistPlaneArgs& a, cudaStream_t st) {
    return dtype == 0 ? run_dist<float>(dist_unpack_kernel<float>, a, st) : run_dist<double>(dist_unpack_kernel<double>, a, st);
}
cudaError_t launch_dist_pack(int dtype, const DistPlaneArgs& a, cudaStream_t st) {
    return dtype == 0 ? run_dist<float>(dist_pack_kernel<float>, a, st) : run_dist<double>(dist_pack_kernel<double>, a, st);
}

template <typename T>
static cudaError_t run(void (*k)(const PlaneArgs), const PlaneArgs& a, cudaStream_t st) {
    const long long n = (long long)a.Nx * a.Ny;
    long long blocks = (n + 255) / 256;
    if (blocks > grid_cap()) blocks = grid_cap();
    k<<<(unsigned)blocks, 256, 0, st>>>(a);
    return cudaGetLastError();
}

cudaError_t launch_unpack_nyquist(int dtype, const PlaneArgs& a, cudaStream_t st) {
    return dtype == 0 ? run<float>(unpack_nyquist_kernel<float>, a, st)
                      : run<double>(unpack_nyquist_kernel<double>, a, st);
}

cudaError_t launch_pack_nyquist(int dtype, const PlaneArgs& a, cudaStream_t st) {
    return dtype == 0 ? run<float>(pack_nyquist_kernel<float>, a, st)
                      : run<double>(pack_nyquist_kernel<double>, a, st);
}

// ---------------------------------------------------------------------------------------------------------
// Pencil layout (reading R17): the spectrum of a px x py rank grid is the slab spectrum
// with p = px whose rows of M+1 entries are cut into py pieces: rank (a, b) holds [Nx][Ny/px][cz_b], cz_b = M/py
// (+1 for the last b: the Nyquist column), blocks concatenated in the order [a][b].  One pass over the array:
// dir = 0: slab rows -> pencil blocks (after the forward transform), dir = 1: pencil blocks -> slab rows.
// ---------------------------------------------------------------------------------------------------------
struct PencilArgs {
    const void* src;
    void* dst;
    long long nrows;          // px * Nx * (Ny/px) rows of M+1 entries
    long long rows_per_a;     // Nx * (Ny/px)
    int M, py, dir;
};

template <typename T>
__global__ void pencil_convert_kernel(const PencilArgs a) {
    using C = cx<T>;
    const int pitch = a.M + 1, c = a.M / a.py;
    const C* src = reinterpret_cast<const C*>(a.src);
    C* dst = reinterpret_cast<C*>(a.dst);
    for (long long row = blockIdx.x; row < a.nrows; row += gridDim.x) {
        const long long ia = row / a.rows_per_a, r = row - ia * a.rows_per_a;     // rank row a, row (kx, ky_l) inside it
        const long long slab = row * pitch;
        const long long blk0 = ia * a.rows_per_a * pitch;                          // start of the blocks (a, 0..py-1)
        for (int k = threadIdx.x; k < pitch; k += blockDim.x) {
            int b = k / c;
            if (b > a.py - 1) b = a.py - 1;
            const int cz = b == a.py - 1 ? c + 1 : c;
            const long long pen = blk0 + (long long)b * a.rows_per_a * c + r * cz + (k - b * c);
            if (a.dir == 0) dst[pen] = src[slab + k];
            else dst[slab + k] = src[pen];
        }
    }
}

cudaError_t launch_pencil_convert(int dtype, const PencilArgs& a, cudaStream_t st) {
    long long blocks = a.nrows < grid_cap() ? a.nrows : grid_cap();
    if (dtype == 0) pencil_convert_kernel<float><<<(unsigned)blocks, 256, 0, st>>>(a);
    else pencil_convert_kernel<double><<<(unsigned)blocks, 256, 0, st>>>(a);
    return cudaGetLastError();
}

}  // namespace fft3d
