// fft_configs.cuh -- which FFT lengths this build has kernels for, and how each is factored.
//
// CfgFor<T, N>::type = FftCfg<N, P, r0, r1, ...>: P points per thread, stage radices r_i (each
// dividing P).  Lengths are 2^a (4..4096), 3*2^a (6..3072), 5*2^a (20..1280) and 7*2^a (28..1792): every extent in
// BASELINE.json's configs (64, 256, 1024, 1536 = 3*2^9, 2048) and their halves for the z pass, plus the radix-5
// and radix-7 families of SURVEY.md 8(f)-4.
#pragma once
#include "fft_core.cuh"

#define FFT3D_FOREACH_N(X) \
    X(4) X(8) X(16) X(32) X(64) X(128) X(256) X(512) X(1024) X(2048) X(4096) \
    X(6) X(12) X(24) X(48) X(96) X(192) X(384) X(768) X(1536) X(3072) \
    X(20) X(40) X(80) X(160) X(320) X(640) X(1280) \
    X(28) X(56) X(112) X(224) X(448) X(896) X(1792)

namespace fft3d {

template <typename T, int N> struct CfgFor;

#define FFT3D_CFG(T_, N_, ...) \
    template <> struct CfgFor<T_, N_> { using type = FftCfg<N_, __VA_ARGS__>; };

// fp32: up to 16 (24 for 3*2^a) points per thread
FFT3D_CFG(float, 4, 4, 4)
FFT3D_CFG(float, 8, 8, 8)
FFT3D_CFG(float, 16, 16, 16)
FFT3D_CFG(float, 32, 8, 8, 4)
FFT3D_CFG(float, 64, 8, 8, 8)
FFT3D_CFG(float, 128, 16, 16, 8)
FFT3D_CFG(float, 256, 16, 16, 16)
FFT3D_CFG(float, 512, 16, 16, 16, 2)
FFT3D_CFG(float, 1024, 32, 32, 32)
FFT3D_CFG(float, 2048, 32, 32, 32, 2)
FFT3D_CFG(float, 4096, 16, 16, 16, 16)
FFT3D_CFG(float, 6, 6, 6)
FFT3D_CFG(float, 12, 12, 12)
FFT3D_CFG(float, 24, 12, 12, 2)
FFT3D_CFG(float, 48, 12, 12, 4)
FFT3D_CFG(float, 96, 12, 12, 4, 2)
FFT3D_CFG(float, 192, 12, 12, 4, 4)
FFT3D_CFG(float, 384, 24, 24, 8, 2)
FFT3D_CFG(float, 768, 24, 24, 8, 4)
FFT3D_CFG(float, 1536, 24, 24, 8, 8)
FFT3D_CFG(float, 3072, 24, 24, 8, 8, 2)

// 5*2^a (radix-5 leaf in fft_radix.cuh)
FFT3D_CFG(float, 20, 20, 20)
FFT3D_CFG(float, 40, 20, 20, 2)
FFT3D_CFG(float, 80, 20, 20, 4)
FFT3D_CFG(float, 160, 20, 20, 4, 2)
FFT3D_CFG(float, 320, 20, 20, 4, 4)
FFT3D_CFG(float, 640, 20, 20, 4, 4, 2)
FFT3D_CFG(float, 1280, 20, 20, 4, 4, 4)

// 7*2^a (radix-7 leaf in fft_radix.cuh)
FFT3D_CFG(float, 28, 28, 28)
FFT3D_CFG(float, 56, 28, 28, 2)
FFT3D_CFG(float, 112, 28, 28, 4)
FFT3D_CFG(float, 224, 28, 28, 4, 2)
FFT3D_CFG(float, 448, 28, 28, 4, 4)
FFT3D_CFG(float, 896, 28, 28, 4, 4, 2)
FFT3D_CFG(float, 1792, 28, 28, 4, 4, 4)

// fp64: registers are twice as wide, so fewer points per thread
FFT3D_CFG(double, 4, 4, 4)
FFT3D_CFG(double, 8, 8, 8)
FFT3D_CFG(double, 16, 16, 16)
FFT3D_CFG(double, 32, 8, 8, 4)
FFT3D_CFG(double, 64, 8, 8, 8)
FFT3D_CFG(double, 128, 8, 8, 8, 2)
FFT3D_CFG(double, 256, 16, 16, 16)
FFT3D_CFG(double, 512, 8, 8, 8, 8)
FFT3D_CFG(double, 1024, 16, 16, 16, 4)
FFT3D_CFG(double, 2048, 16, 16, 16, 8)
FFT3D_CFG(double, 4096, 16, 16, 16, 16)
FFT3D_CFG(double, 6, 6, 6)
FFT3D_CFG(double, 12, 12, 12)
FFT3D_CFG(double, 24, 12, 12, 2)
FFT3D_CFG(double, 48, 12, 12, 4)
FFT3D_CFG(double, 96, 12, 12, 4, 2)
FFT3D_CFG(double, 192, 12, 12, 4, 4)
FFT3D_CFG(double, 384, 12, 12, 4, 4, 2)
FFT3D_CFG(double, 768, 12, 12, 4, 4, 4)
FFT3D_CFG(double, 1536, 12, 12, 4, 4, 4, 2)
FFT3D_CFG(double, 3072, 12, 12, 4, 4, 4, 4)

FFT3D_CFG(double, 20, 20, 20)
FFT3D_CFG(double, 40, 20, 20, 2)
FFT3D_CFG(double, 80, 20, 20, 4)
FFT3D_CFG(double, 160, 20, 20, 4, 2)
FFT3D_CFG(double, 320, 20, 20, 4, 4)
FFT3D_CFG(double, 640, 20, 20, 4, 4, 2)
FFT3D_CFG(double, 1280, 20, 20, 4, 4, 4)

FFT3D_CFG(double, 28, 28, 28)
FFT3D_CFG(double, 56, 28, 28, 2)
FFT3D_CFG(double, 112, 28, 28, 4)
FFT3D_CFG(double, 224, 28, 28, 4, 2)
FFT3D_CFG(double, 448, 28, 28, 4, 4)
FFT3D_CFG(double, 896, 28, 28, 4, 4, 2)
FFT3D_CFG(double, 1792, 28, 28, 4, 4, 4)

// Factorisation used by the bulk-pipelined z kernels (fft_zpass.cuh): the strided-pass one unless
// a shape with fewer exchanges fits a row's threads inside one warp.
template <typename T, int N> struct ZCfgFor { using type = typename CfgFor<T, N>::type; };
template <> struct ZCfgFor<float, 512> { using type = FftCfg<512, 32, 32, 16>; };
template <> struct ZCfgFor<float, 256> { using type = FftCfg<256, 16, 16, 16>; };
// fp64 512 = 32*16: one exchange instead of two, 128 data registers per thread in 128-thread groups
// (1024^3 fp64: z_r2c 3.41 -> 2.90 ms; 16*16*2 before)
template <> struct ZCfgFor<double, 512> { using type = FftCfg<512, 32, 32, 16>; };
// 768 = 48*16: one exchange instead of two (the z passes are shared-memory bound: 0.73 wavefronts per cycle per SM);
// 48 points per thread need one 256-thread group with 224 registers instead of two with 120
template <> struct ZCfgFor<float, 768> { using type = FftCfg<768, 48, 48, 16>; };

// Tile width (columns) of the strided passes: 128-byte rows while the tile stays small,
// 64-byte rows up to N = 2048, 32-byte rows beyond.
__host__ __device__ constexpr int tile_cols(int N, int csize) {
    int row_bytes = N <= 256 ? 128 : (N <= 2048 ? 64 : 32);
    return row_bytes / csize;
}

// Tile width of the TMA-pipelined strided passes (0 = not built for this length): the consumer
// count S*TC must be a multiple of 32 and leave room for the producer warp.
__host__ __device__ constexpr int tma_tile_cols(int N, int S, int csize) {
    int tc = tile_cols(N, csize);
    while (tc > 1 && S * tc + 32 > 1024) tc /= 2;
    if (tc * csize < 32) return 0;                 // rows narrower than a sector: not worth it
    if ((S * tc) % 32 != 0 || N < 64) return 0;
    return tc;
}

// Rows per CTA iteration of the z passes: aim for ~256 threads.
__host__ __device__ constexpr int rows_per_block(int S) {
    int r = 256 / S;
    return r < 1 ? 1 : (r > 16 ? 16 : r);
}

// Resident CTAs per SM the kernels are compiled for (register cap via __launch_bounds__).
__host__ __device__ constexpr int min_blocks(int threads, int P, int tsize, size_t smem) {
    int need = P * 2 * (tsize / 4) + 32;                  // data registers + working set
    if (need > 255) need = 255;
    int by_regs = 65536 / (threads * need);
    int by_thr = 2048 / threads;
    int by_smem = (int)((227 * 1024) / (smem + 1024));
    int b = by_regs < by_thr ? by_regs : by_thr;
    b = b < by_smem ? b : by_smem;
    return b < 1 ? 1 : (b > 8 ? 8 : b);
}

}  // namespace fft3d
