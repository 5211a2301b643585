// fft_inst.cu -- compiled once per FFT length (-DFFT3D_N=<n>): instantiates the z and strided
// kernels for fp32 and fp64 and exports their description.
#include "fft_kernels.cuh"
#include "fft_zpass.cuh"
#include "fft_fused.cuh"
#include "fft_split2.cuh"
#include "fft_configs.cuh"
#include "fft_registry.h"

#ifndef FFT3D_N
#error "compile with -DFFT3D_N=<length>"
#endif

namespace fft3d {

// fused z+y kernels for Nz == Ny == N (z FFT of N/2 points, y FFT of N points)
template <typename T, int N>
static void add_fused(KernelSet& k) {
    if constexpr (N >= 128) {
        using C = cx<T>;
        using YCfg = typename CfgFor<T, N>::type;
        using ZCfg = typename ZCfgFor<T, N / 2>::type;
        constexpr int TTC = tma_tile_cols(YCfg::N, YCfg::S, (int)sizeof(C));
        if constexpr (TTC > 0 && ZCfg::S >= 8 && ZCfg::S <= 32 && (ZCfg::S & (ZCfg::S - 1)) == 0 && ZCfg::P % 2 == 0 &&
                      (YCfg::S * TTC) % ZCfg::S == 0) {
            constexpr int RPT = YCfg::S * TTC / ZCfg::S;
            constexpr int GROUP = YCfg::S * TTC;
            constexpr int NG = (2 * GROUP + 64 <= 1024 && FusedTile<ZCfg, RPT, YCfg, TTC, T, 2>::max_stages() >= 3) ? 2 : 1;
            using FT = FusedTile<ZCfg, RPT, YCfg, TTC, T, NG>;
            constexpr int NS = FT::max_stages();
            if constexpr (FT::OK && NS >= 2 && FT::THREADS <= 1024) {
                k.fz_fn[0] = (const void*)fft_zy_fused_kernel<ZCfg, RPT, YCfg, TTC, -1, T, NS, NG>;
                k.fz_fn[1] = (const void*)fft_zy_fused_kernel<ZCfg, RPT, YCfg, TTC, +1, T, NS, NG>;
                k.fz_rpt = RPT;
                k.fz_tc = TTC;
                k.fz_threads = FT::THREADS;
                k.fz_smem = (size_t)FT::smem_bytes(NS);
                k.fz_ng = NG;
                k.fz_nstage = NS;
            }
        }
    }
}

// Y passes of length N as two N/2-point half tiles (only where the whole tile leaves room for one ring stage)
template <typename T, int N>
static void add_split2(KernelSet& k) {
    if constexpr (N >= 256 && N % 2 == 0) {
        using C = cx<T>;
        using Cfg = typename CfgFor<T, N>::type;
        using HCfg = typename CfgFor<T, N / 2>::type;
        constexpr int TTC = tma_tile_cols(Cfg::N, Cfg::S, (int)sizeof(C));
        constexpr int HTC = tma_tile_cols(HCfg::N, HCfg::S, (int)sizeof(C));
        if constexpr (TTC > 0 && HTC == TTC) {
            using TY = TmaTile<Cfg, TTC, T, false>;
            using TH = TmaTile<HCfg, TTC, T, false>;
            k.y2_nst = HCfg::NST;
            for (int s = 0; s < 5; ++s) k.y2_radix[s] = s < HCfg::NST ? HCfg::radix(s) : 1;
            k.y2_twn = HCfg::TWN;
            if constexpr (TY::max_stages() <= 1 && TH::max_stages() >= 3) {
                constexpr int NS = 3;
                k.y2_fn[0] = (const void*)fft_y_split2_kernel<HCfg, TTC, TMA_Y_FWD, T, NS>;
                k.y2_fn[1] = (const void*)fft_y_split2_kernel<HCfg, TTC, TMA_Y_INV, T, NS>;
                k.y2_threads = TH::NCONS + 32;
                k.y2_smem = (size_t)TH::smem_bytes(NS);
            }
            using TXW = TmaTile<Cfg, TTC, T, true>;
            using THW = TmaTile<HCfg, TTC, T, true>;
            if constexpr (TXW::max_stages() <= 1 && THW::max_stages() >= 3) {
                constexpr int NS = 3;
                k.x2_fn[0] = (const void*)fft_x_split2_kernel<HCfg, TTC, TMA_X_FWD, T, NS>;
                k.x2_fn[1] = (const void*)fft_x_split2_kernel<HCfg, TTC, TMA_X_INV, T, NS>;
                k.x2_threads = THW::NCONS + 32;
                k.x2_smem = (size_t)THW::smem_bytes(NS);
            }
        }
    }
}

// X passes of length N as four N/4-point quarter tiles (where neither the whole nor the half tile pipelines)
template <typename T, int N>
static void add_split4(KernelSet& k) {
    if constexpr (N >= 1024 && N % 4 == 0) {
        using C = cx<T>;
        using Cfg = typename CfgFor<T, N>::type;
        using HCfg = typename CfgFor<T, N / 2>::type;
        using QCfg = typename CfgFor<T, N / 4>::type;
        constexpr int TTC = tma_tile_cols(Cfg::N, Cfg::S, (int)sizeof(C));
        constexpr int QTC = tma_tile_cols(QCfg::N, QCfg::S, (int)sizeof(C));
        if constexpr (TTC > 0 && QTC == TTC) {
            using TXW = TmaTile<Cfg, TTC, T, true>;
            using THW = TmaTile<HCfg, TTC, T, true>;
            using TQW = TmaTile<QCfg, TTC, T, true>;
            constexpr int NS = 5;
            if constexpr (TXW::max_stages() <= 1 && THW::max_stages() < 3 && TQW::smem_bytes(NS) <= 227 * 1024) {
                k.x4_fn[0] = (const void*)fft_x_split4_kernel<QCfg, TTC, TMA_X_FWD, T, NS>;
                k.x4_fn[1] = (const void*)fft_x_split4_kernel<QCfg, TTC, TMA_X_INV, T, NS>;
                k.x4_threads = TQW::NCONS + 32;
                k.x4_smem = (size_t)TQW::smem_bytes(NS);
                k.x4_nst = QCfg::NST;
                for (int s = 0; s < 5; ++s) k.x4_radix[s] = s < QCfg::NST ? QCfg::radix(s) : 1;
                k.x4_twn = QCfg::TWN;
            }
        }
    }
}

// fused z+y kernels of C2C plans with Nz == Ny == N
template <typename T, int N>
static void add_fused_c2c(KernelSet& k) {
    if constexpr (N >= 128) {
        using C = cx<T>;
        using YCfg = typename CfgFor<T, N>::type;
        using ZCfg = typename ZCfgFor<T, N>::type;
        constexpr int TTC = tma_tile_cols(YCfg::N, YCfg::S, (int)sizeof(C));
        if constexpr (TTC > 0 && (YCfg::S * TTC) % ZCfg::S == 0 && ZCfg::S <= YCfg::S * TTC) {
            constexpr int RPT = YCfg::S * TTC / ZCfg::S;
            constexpr int GROUP = YCfg::S * TTC;
            constexpr int NG = (2 * GROUP + 128 <= 1024 && FusedTile<ZCfg, RPT, YCfg, TTC, T, 2>::max_stages() >= 3) ? 2 : 1;
            using FT = FusedTile<ZCfg, RPT, YCfg, TTC, T, NG>;
            constexpr int NS = FT::max_stages();
            if constexpr (FT::OK && NS >= 3 && NG >= 2 && FT::THREADS <= 1024) {      // only where fusion can win
                k.fc_fn[0] = (const void*)fft_zy_fused_kernel<ZCfg, RPT, YCfg, TTC, -1, T, NS, NG, true>;
                k.fc_fn[1] = (const void*)fft_zy_fused_kernel<ZCfg, RPT, YCfg, TTC, +1, T, NS, NG, true>;
                k.fc_rpt = RPT; k.fc_tc = TTC; k.fc_threads = FT::THREADS; k.fc_smem = (size_t)FT::smem_bytes(NS);
                k.fc_ng = NG; k.fc_nstage = NS;
            }
        }
    }
}

template <typename T>
static KernelSet make_set(int dtype) {
    using Cfg = typename CfgFor<T, FFT3D_N>::type;
    using C = cx<T>;
    constexpr int TC = tile_cols(Cfg::N, (int)sizeof(C));
    using TP = TilePad<Cfg, TC * (int)sizeof(C)>;
    constexpr size_t TWB = (size_t)((Cfg::TWN + 1) & ~1) * sizeof(C);
    constexpr size_t S_SMEM = TWB + (size_t)TP::ROWS * TC * sizeof(C);
    constexpr int S_THREADS = Cfg::S * TC;
    // the second register set of the prefetching variant must fit the register file
    constexpr bool S_PF = (S_THREADS * (4 * Cfg::P * (int)sizeof(T) / 4 + 48) <= 65536);
    constexpr int S_MINB = S_PF ? 1 : min_blocks(S_THREADS, Cfg::P, (int)sizeof(T), S_SMEM);
    constexpr int RPB = rows_per_block(Cfg::S);
    constexpr size_t Z_SMEM = TWB + (size_t)Cfg::N * sizeof(C) + (size_t)RPB * RowPad<Cfg>::PITCH * sizeof(C);
    constexpr int Z_THREADS = Cfg::S * RPB;
    constexpr int Z_MINB = min_blocks(Z_THREADS, Cfg::P, (int)sizeof(T), Z_SMEM);

    KernelSet k{};
    k.N = Cfg::N;
    k.dtype = dtype;
    k.P = Cfg::P;
    k.nst = Cfg::NST;
    for (int s = 0; s < 5; ++s) k.radix[s] = s < Cfg::NST ? Cfg::radix(s) : 1;
    k.twn = Cfg::TWN;
    k.tc = TC;
    k.s_threads = S_THREADS;
    k.s_smem = S_SMEM;
    k.s_fn[0][KIND_LIN_LIN]  = (const void*)fft_strided_kernel<Cfg, TC, -1, false, false, T, S_MINB, S_PF>;
    k.s_fn[0][KIND_LIN_SLAB] = (const void*)fft_strided_kernel<Cfg, TC, -1, false, true, T, S_MINB, S_PF>;
    k.s_fn[0][KIND_SLAB_LIN] = nullptr;
    k.s_fn[1][KIND_LIN_LIN]  = (const void*)fft_strided_kernel<Cfg, TC, +1, false, false, T, S_MINB, S_PF>;
    k.s_fn[1][KIND_LIN_SLAB] = nullptr;
    k.s_fn[1][KIND_SLAB_LIN] = (const void*)fft_strided_kernel<Cfg, TC, +1, true, false, T, S_MINB, S_PF>;
    k.z_rpb = RPB;
    k.z_threads = Z_THREADS;
    k.z_smem = Z_SMEM;
    k.z_fn[0] = (const void*)fft_z_r2c_kernel<Cfg, RPB, T, Z_MINB>;
    k.z_fn[1] = (const void*)fft_z_c2r_kernel<Cfg, RPB, T, Z_MINB>;
    k.zp_fn[0] = (const void*)fft_z_c2c_kernel<Cfg, RPB, -1, T, Z_MINB>;
    k.zp_fn[1] = (const void*)fft_z_c2c_kernel<Cfg, RPB, +1, T, Z_MINB>;
    constexpr int TTC = tma_tile_cols(Cfg::N, Cfg::S, (int)sizeof(C));
    if constexpr (TTC > 0) {
        // complex fp32 rows of the user's spectrum (M+1 entries) start on 8-byte boundaries for odd l:
        // the X passes shift those tiles' windows (ODDFIX, see fft_kernels.cuh)
        // (fp64: the same shift puts the 64-byte windows of odd rows on 32-byte sectors of the user array)
        constexpr bool OF = true;
        using TY = TmaTile<Cfg, TTC, T, false>;
        // X passes: same tile width (48-byte rows were tried to get a second ring stage back at
        // N = 1536 where the shifted windows land TC+2 columns: rows that are not a multiple of the
        // 32-byte sector cost 2.5x, measured)
        constexpr int TTCX = TTC;
        using TX = TmaTile<Cfg, TTCX, T, OF>;
        constexpr int NSY = TY::max_stages(), NSX = TX::max_stages();
        // one ring stage still works (load, transform, store in turn; the other SMs keep HBM busy)
        if constexpr (NSY >= 1) {
            k.tma_fn[TMA_Y_FWD] = (const void*)fft_strided_tma_kernel<Cfg, TTC, TMA_Y_FWD, T, NSY, false>;
            k.tma_fn[TMA_Y_INV] = (const void*)fft_strided_tma_kernel<Cfg, TTC, TMA_Y_INV, T, NSY, false>;
            k.tma_smem_y = (size_t)TY::smem_bytes(NSY);
        }
        if constexpr (NSX >= 1) {
            k.tma_fn[TMA_X_FWD] = (const void*)fft_strided_tma_kernel<Cfg, TTCX, TMA_X_FWD, T, NSX, OF>;
            k.tma_fn[TMA_X_INV] = (const void*)fft_strided_tma_kernel<Cfg, TTCX, TMA_X_INV, T, NSX, OF>;
            k.tma_smem_x = (size_t)TX::smem_bytes(NSX);
        }
        {   // C2C plans: both sides of the x pass have pitch Nz (aligned rows): the plain windows
            using TXC = TmaTile<Cfg, TTCX, T, false>;
            constexpr int NSC = TXC::max_stages();
            if constexpr (NSC >= 1) {
                k.xc_fn[0] = (const void*)fft_strided_tma_kernel<Cfg, TTCX, TMA_X_FWD, T, NSC, false>;
                k.xc_fn[1] = (const void*)fft_strided_tma_kernel<Cfg, TTCX, TMA_X_INV, T, NSC, false>;
                k.xc_smem = (size_t)TXC::smem_bytes(NSC);
            }
        }
        k.tma_oddfix = OF ? 1 : 0;
        k.tma_tc = TTC;
        k.tma_threads = TY::NCONS + 32;
        k.tma_tc_x = TTCX;
        k.tma_threads_x = TX::NCONS + 32;
    }
    // bulk-pipelined z kernels: a row's S threads inside one warp, ~256 threads per 64 KiB tile
    using ZCfg = typename ZCfgFor<T, FFT3D_N>::type;
    if constexpr (ZCfg::S >= 8 && ZCfg::S <= 32 && (ZCfg::S & (ZCfg::S - 1)) == 0 && ZCfg::P % 2 == 0 &&
                  ZCfg::N * sizeof(C) >= 1024) {
        // fp64: 128 threads per tile (two groups + producer = 288 threads, 224 registers each: with 256-thread groups
        // the 120-register cap made the fp64 C2R kernel spill 184 bytes per thread)
        constexpr int GRP = sizeof(T) == 8 && ZCfg::S <= 16 * 8 && 128 % ZCfg::S == 0 ? 128 : 256;
        constexpr int RPT = GRP / ZCfg::S;
        using ZT = ZTile<ZCfg, RPT, T>;
        constexpr int NG = (ZT::max_stages(2) >= 3 && ZCfg::P <= 32) ? 2 : 1;      // P > 32: one group, 224 registers
        constexpr int NS = ZT::max_stages(NG) > 4 ? 4 : ZT::max_stages(NG);
        if constexpr (NS >= 2) {
            k.zb_fn[0] = (const void*)fft_z_bulk_kernel<ZCfg, RPT, -1, T, NS, NG>;
            k.zb_fn[1] = (const void*)fft_z_bulk_kernel<ZCfg, RPT, +1, T, NS, NG>;
            k.zb_rpt = RPT;
            k.zb_nst = ZCfg::NST;
            for (int s = 0; s < 5; ++s) k.zb_radix[s] = s < ZCfg::NST ? ZCfg::radix(s) : 1;
            k.zb_twn = ZCfg::TWN;
            k.zb_threads = ZT::GROUP * NG + 32;
            k.zb_smem = (size_t)ZT::smem_bytes(NS, NG);
        }
    }
    // C2C row kernels: 256 threads per tile of 256/S rows, any S that divides 256
    if constexpr (ZCfg::S <= 256 && 256 % ZCfg::S == 0 && ZCfg::N * sizeof(C) >= 1024) {
        constexpr int RPT = 256 / ZCfg::S;
        using ZT = ZTile<ZCfg, RPT, T>;
        constexpr int NG = ZT::max_stages(2) >= 3 ? 2 : 1;
        constexpr int NS = ZT::max_stages(NG) > 4 ? 4 : ZT::max_stages(NG);
        if constexpr (NS >= 2) {
            k.zc_fn[0] = (const void*)fft_z_bulk_kernel<ZCfg, RPT, -1, T, NS, NG, true>;
            k.zc_fn[1] = (const void*)fft_z_bulk_kernel<ZCfg, RPT, +1, T, NS, NG, true>;
            k.zc_rpt = RPT;
            k.zc_nst = ZCfg::NST;
            for (int s = 0; s < 5; ++s) k.zc_radix[s] = s < ZCfg::NST ? ZCfg::radix(s) : 1;
            k.zc_twn = ZCfg::TWN;
            k.zc_threads = ZT::GROUP * NG + 32;
            k.zc_smem = (size_t)ZT::smem_bytes(NS, NG);
        }
    }
    add_fused<T, FFT3D_N>(k);
    add_fused_c2c<T, FFT3D_N>(k);
    add_split2<T, FFT3D_N>(k);
    add_split4<T, FFT3D_N>(k);
    return k;
}

#define FFT3D_CAT2(a, b) a##b
#define FFT3D_CAT(a, b) FFT3D_CAT2(a, b)

const KernelSet* FFT3D_CAT(kernelset_, FFT3D_N)(int dtype) {
    static const KernelSet f32 = make_set<float>(0);
    static const KernelSet f64 = make_set<double>(1);
    return dtype == 0 ? &f32 : &f64;
}

}  // namespace fft3d
