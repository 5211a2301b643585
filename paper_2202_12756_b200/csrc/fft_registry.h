// fft_registry.h -- host-side description of the kernels compiled for one FFT length and dtype.
#pragma once
#include <cstddef>

namespace fft3d {

enum { KIND_LIN_LIN = 0, KIND_LIN_SLAB = 1, KIND_SLAB_LIN = 2 };

struct KernelSet {
    int N;                 // FFT length (for the z kernels: M = Nz/2)
    int dtype;             // FFT3D_F32 / FFT3D_F64
    int P;                 // points per thread
    int nst;               // stages
    int radix[5];
    int twn;               // stage-twiddle table entries
    // strided C2C kernels (N rows x TC columns per tile)
    int tc;
    int s_threads;
    size_t s_smem;
    const void* s_fn[2][3];    // [0 = forward, 1 = inverse][kind]; null if not compiled
    // z kernels (rows of N packed complex)
    int z_rpb;
    int z_threads;
    size_t z_smem;
    const void* z_fn[2];       // [0 = R2C, 1 = C2R]
    const void* zp_fn[2];      // plain-load C2C row kernels [0 = forward, 1 = inverse (scaled)]: same launch shape
    // TMA-pipelined strided kernels (null if not compiled for this length)
    const void* tma_fn[4];     // [TMA_Y_FWD, TMA_Y_INV, TMA_X_FWD, TMA_X_INV]
    int tma_tc;                // tile columns of the Y passes
    int tma_threads;           // consumers + one producer warp
    int tma_tc_x;              // tile columns / threads of the X passes (narrower when the shifted windows need room)
    int tma_threads_x;
    int tma_oddfix;            // 1: the X passes shift the windows of odd-l rows (fp32, see fft_kernels.cuh)
    size_t tma_smem_y, tma_smem_x;
    // bulk-copy pipelined z kernels (null if not compiled for this length)
    const void* zb_fn[2];      // [0 = R2C, 1 = C2R]
    int zb_rpt;                // rows per tile: the row count must be a multiple
    int zb_nst, zb_radix[5], zb_twn;   // their factorisation (it may differ from the strided kernels')
    int zb_threads;            // consumer groups + one producer warp
    size_t zb_smem;
    // TMA-pipelined X kernels for layouts whose two sides share one aligned pitch (C2C plans): no shifted windows
    const void* xc_fn[2];      // [0 = X_FWD, 1 = X_INV]
    size_t xc_smem;
    // Y passes as two half tiles + one radix-2 combine (fft_split2.cuh); null unless the whole tile has a single stage
    const void* y2_fn[2];      // [0 = Y_FWD, 1 = Y_INV]
    int y2_threads, y2_nst, y2_radix[5], y2_twn;   // y2_nst.. = the factorisation of the N/2-point transform (X kernels too)
    size_t y2_smem;
    const void* x2_fn[2];      // the same for the X passes with shifted windows: [0 = X_FWD, 1 = X_INV]
    int x2_threads;
    size_t x2_smem;
    const void* x4_fn[2];      // X passes as four quarter tiles + a radix-4 combine
    int x4_threads, x4_nst, x4_radix[5], x4_twn;   // x4_nst.. = the factorisation of the N/4-point transform
    size_t x4_smem;
    // C2C row kernels (z pass of the 3D C2C transform): the bulk-pipelined kernel without the Hermitian step
    const void* zc_fn[2];      // [0 = forward, 1 = inverse (scaled)]
    int zc_rpt, zc_nst, zc_radix[5], zc_twn, zc_threads;
    size_t zc_smem;
    // fused z+y kernels of a cubic-like plan (Nz == Ny == N): fft_fused.cuh; null if not compiled
    const void* fz_fn[2];      // [0 = F1+F2, 1 = I2+I3]
    int fz_rpt;                // rows per z tile (Ny must be a multiple)
    int fz_tc;                 // columns per y tile (Nz/2 must be a multiple)
    int fz_threads;
    size_t fz_smem;
    int fz_ng, fz_nstage;      // consumer groups per CTA, shared-memory ring depth
    // the same for C2C plans (Nz == Ny == N: rows of N complex points)
    const void* fc_fn[2];
    int fc_rpt, fc_tc, fc_threads, fc_ng, fc_nstage;
    size_t fc_smem;
};

// nullptr if this build has no kernels for (n, dtype)
const KernelSet* find_kernels(long long n, int dtype);

}  // namespace fft3d
