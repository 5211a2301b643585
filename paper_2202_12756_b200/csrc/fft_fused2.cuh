// fft_fused2.cuh -- second generation of the fused z+y passes:
//
//   fft_zy_fused2_kernel<DIR = -1>  passes F1+F2 of every x-plane in ONE persistent kernel: z-axis R2C of the
//                                   plane's rows (paper step 1, z half) -> ring in L2 -> y-axis C2C with
//                                   each row ky written to its slab address (step 1 y half + steps 2-4)
//   fft_zy_fused2_kernel<DIR = +1>  passes I2+I3, the mirror image, 1/(NxNyNz) fused
//
// The dataflow between CTAs is that of fft_fused.cuh (roles per SM, column-tiled ring [R][M/TC][Ny][TC] that
// stays in L2, two counters per plane).  What changes is the pipeline INSIDE a CTA.  The first generation
// transformed a tile in place in one of three 67 KiB ring slots; two slots were held by the two consumer
// groups for the whole transform, so a single tile was in flight per SM and the consumers waited for tiles
// ~40 % of the time (profiles/r1_k_ncu_full.md: 36 % of the samples on the mbarrier poll of full[]).
// Here a tile's life is split between three kinds of storage:
//
//   landing buffer  one dense tile (64 KiB) filled by TMA in two halves; a consumer group copies a landed
//                   half into REGISTERS and hands it straight back, so the next tile's loads run during the
//                   whole transform of this one;
//   registers       the group's threads hold the tile (P points each) through the first butterfly stage;
//   work buffer     one per group: the exchange between the butterfly stages, then the dense output tile the
//                   group's store thread hands to TMA.  The group starts its NEXT tile (landing -> registers ->
//                   first stage) while that store is still draining, and only waits for the work buffer to be
//                   free before the exchange.
//
// Loads are therefore hidden behind a whole tile of arithmetic and stores behind the first stage of the next
// tile, with the same shared memory (64 + 2 x 67 KiB) as three in-place slots.
//
// Roles and ranks: a CTA takes the z tiles or the y tiles for the whole launch (the two tile bodies are ~35 KB
// of straight-line code each and the two SMs of a TPC share an instruction cache: with both bodies alive in a
// TPC 60 % of the issue stalls were instruction fetches).  The role follows %smid (SMs [0, kz) -> z), but
// nothing is assumed about the ids being dense or one CTA per SM: every CTA draws its rank inside its role
// from an atomic ticket and learns the role sizes after a grid-wide arrival counter (cooperative launch: all
// CTAs are co-resident).  If a role came out empty, all CTAs fall back to a split by blockIdx.
//
// Every spin on a global counter is bounded: a kernel that cannot make progress traps (the host then sees a
// launch failure and the API returns FFT3D_ECUDA) instead of hanging the device.
#pragma once
#include <cstdint>

#include "fft_core.cuh"
#include "fft_kernels.cuh"
#include "fft_zpass.cuh"
#include "fft_fused.cuh"

namespace fft3d {

// words of the control block that follows the 2*Nx plane counters in the flags area
enum { FZ_CTL_NZ = 0, FZ_CTL_NY = 1, FZ_CTL_ARRIVED = 2, FZ_CTL_WORDS = 8 };

namespace tma {
// bounded spin on a global counter (see the header comment): ~1 us per poll, 2^24 polls > 10 s
__device__ __forceinline__ void wait_count_bounded(const unsigned* p, unsigned target) {
    unsigned polls = 0;
    while (ld_acquire(p) < target) {
        __nanosleep(64);
        if (++polls > (1u << 24)) __trap();
    }
}
}  // namespace tma

template <class ZCfg, int RPT, class YCfg, int TC, typename T, int NG_ = 2>
struct Fused2Tile {
    using C = cx<T>;
    using ZT = ZTile<ZCfg, RPT, T>;
    using YT = TmaTile<YCfg, TC, T, false>;
    static constexpr int GROUP = ZT::GROUP;                     // consumer threads per group
    static constexpr int NG = NG_;
    static constexpr bool OK = (ZT::GROUP == YT::NCONS) && (ZT::GROUP % 64 == 0) && (RPT % 2 == 0) &&
                               (ZT::TILE_BYTES % 2048 == 0) && (YT::TILE_BYTES % 2048 == 0) && (YCfg::P % 2 == 0);
    static constexpr int WORK_BYTES = ZT::STAGE_BYTES > YT::STAGE_BYTES ? ZT::STAGE_BYTES : YT::STAGE_BYTES;
    static constexpr int LAND_BYTES = ZT::TILE_BYTES > YT::TILE_BYTES ? ZT::TILE_BYTES : YT::TILE_BYTES;
    static constexpr int TW_BYTES = ZT::TW_BYTES > YT::TW_BYTES ? ZT::TW_BYTES : YT::TW_BYTES;   // one role per CTA
    static constexpr int SCRATCH_BYTES = NG * ZT::SCRATCH_BYTES;
    static constexpr int SMEM_BYTES = TW_BYTES + LAND_BYTES + NG * WORK_BYTES + SCRATCH_BYTES + 256;
    // consumer groups + one load warp + one store warp per group
    static constexpr int THREADS = NG * GROUP + 32 * (1 + NG);
    static constexpr bool FITS = SMEM_BYTES <= 227 * 1024 && THREADS <= 1024;
};

// Read elements t + m*S, m in [M0, M1), of the thread's column / row from a dense tile.
template <class Cfg, int M0, int M1, typename T, class Lay>
__device__ __forceinline__ void read_own_range(cx<T> (&v)[Cfg::P], const cx<T>* __restrict__ sm, int t, const Lay& lay) {
    static_assert(Lay::PADR == 0, "dense layout");
    const cx<T>* b = sm + lay.at(t);
#pragma unroll
    for (int m = M0; m < M1; ++m) v[m] = b[Lay::off(m * Cfg::S)];
}

// C2C = true: the rows are Nz complex numbers and the z tiles run the plain C2C transform (3D C2C plans)
template <class ZCfg, int RPT, class YCfg, int TC, int DIR, typename T, int NG_, bool C2C = false>
__global__ void __launch_bounds__((Fused2Tile<ZCfg, RPT, YCfg, TC, T, NG_>::THREADS), 1)
fft_zy_fused2_kernel(const __grid_constant__ TensorMapBlob ring_map, const __grid_constant__ TensorMapBlob slab_map,
                     const FusedArgs a) {
    using C = cx<T>;
    using FT = Fused2Tile<ZCfg, RPT, YCfg, TC, T, NG_>;
    using ZT = typename FT::ZT;
    using YT = typename FT::YT;
    constexpr int GROUP = FT::GROUP, NG = FT::NG, NCONS = NG * GROUP, W = YT::W;
    constexpr int M = ZCfg::N, NY = YCfg::N;
    constexpr bool FWD = DIR < 0;
    static_assert(FT::OK, "z tile and y tile must use the same number of consumer threads; whole halves");
    static_assert(C2C || (ZCfg::S <= 32 && (ZCfg::S & (ZCfg::S - 1)) == 0), "a row's threads must sit inside one warp");

    extern __shared__ __align__(1024) unsigned char smem_dyn[];
    C* tw_s = reinterpret_cast<C*>(smem_dyn);                                    // this role's stage twiddles
    unsigned char* land = smem_dyn + FT::TW_BYTES;                               // one dense tile, two halves
    unsigned char* work = land + FT::LAND_BYTES;                                 // NG work buffers
    C* scratch = reinterpret_cast<C*>(work + NG * FT::WORK_BYTES);
    unsigned long long* full = reinterpret_cast<unsigned long long*>(reinterpret_cast<unsigned char*>(scratch) + FT::SCRATCH_BYTES);
    unsigned long long* empty = full + 2;                // consumers -> load thread: half read into registers
    unsigned long long* wdone = empty + 2;               // group -> its store thread: output tile complete
    unsigned long long* wfree = wdone + NG;              // store thread -> group: work buffer read out
    // turn = index of the CTA's tile whose landing may be awaited.  The two groups use full[] in turn and a
    // parity wait only tells the barrier's current phase from the one before it, so a group must not start
    // waiting for tile i before the phase of tile i-1 has been observed complete.
    volatile int* turn = reinterpret_cast<volatile int*>(wfree + NG);
    volatile int* role_s = turn + 1;                     // [role_z, rank, nrole] broadcast from thread 0

    const int tid = threadIdx.x;
    unsigned* p1_done = a.flags;
    unsigned* p2_loaded = a.flags + a.Nx;
    unsigned* ctl = a.flags + 2 * a.Nx;

    // ---- role and rank (see the header comment) ----
    if (tid == 0) {
        unsigned smid;
        asm("mov.u32 %0, %%smid;" : "=r"(smid));
        const int b = blockIdx.x, G = gridDim.x;
        int role_z = (a.kz > 0 && a.kz < G) ? ((int)smid < a.kz) : !((b >> 1) & 1);
        int rank = (int)atomicAdd(&ctl[role_z ? FZ_CTL_NZ : FZ_CTL_NY], 1u);
        __threadfence();
        tma::red_release_add(&ctl[FZ_CTL_ARRIVED], 1u);
        tma::wait_count_bounded(&ctl[FZ_CTL_ARRIVED], (unsigned)G);
        int nz = (int)tma::ld_acquire(&ctl[FZ_CTL_NZ]), ny = (int)tma::ld_acquire(&ctl[FZ_CTL_NY]);
        int nrole = role_z ? nz : ny;
        if (nz == 0 || ny == 0) {                        // a role came out empty: split by blockIdx instead
            role_z = !(b & 1);
            rank = b >> 1;
            nrole = role_z ? (G + 1) / 2 : G / 2;
        }
        role_s[0] = role_z; role_s[1] = rank; role_s[2] = nrole;
    }
    __syncthreads();
    const int role_z = role_s[0], rank = role_s[1], nrole = role_s[2];

    if (tid == NCONS) {
        for (int h = 0; h < 2; ++h) {
            tma::mbar_init(&full[h], 1);
            // a z tile's half is read by half of the group's warps, a y tile's half by all of them
            tma::mbar_init(&empty[h], role_z ? GROUP / 64 : GROUP / 32);
        }
        for (int g = 0; g < NG; ++g) { tma::mbar_init(&wdone[g], GROUP / 32); tma::mbar_init(&wfree[g], 1); }
        *turn = 0;
        tma::fence_mbar_init();
    }
    if (tid < NCONS) {
        if (role_z) load_twiddles<DIR, T>(tw_s, reinterpret_cast<const C*>(a.tw_z), ZCfg::TWN, tid, NCONS);
        else load_twiddles<DIR, T>(tw_s, reinterpret_cast<const C*>(a.tw_y), YCfg::TWN, tid, NCONS);
    }
    __syncthreads();

    const int n_z = a.Ny / RPT, n_y = M / TC;            // z tiles / y tiles per plane
    const int n1 = FWD ? n_z : n_y, n2 = FWD ? n_y : n_z;
    const int my_p1 = FWD ? role_z : !role_z;            // this CTA's tiles are the phase-1 tiles
    const int nper = role_z ? n_z : n_y;                 // tiles per plane of this role
    const int total = a.Nx * nper;
    const long long plane_bytes = (long long)a.Ny * M * (long long)sizeof(C);
    constexpr int CHUNK = 16384;                         // bytes per 1-D bulk copy

    if (tid >= NCONS) {
        if (tid == NCONS) {
            // ------------------------- load thread -------------------------
            const unsigned long long pol_stream = tma::policy_evict_first(), pol_keep = tma::policy_evict_last();
            int i = 0, ready = -1;                       // planes <= ready are known to be complete in the ring
            for (int g = rank; g < total; g += nrole, ++i) {
                const int x = g / nper, j = g - x * nper;
                if (!my_p1 && x > ready) {
                    tma::wait_count_bounded(&p1_done[x], (unsigned)n1);
                    tma::fence_proxy_async_all();
                    ready = x;
                }
                for (int h = 0; h < 2; ++h) {
                    if (i > 0) tma::mbar_wait(&empty[h], (unsigned)((i - 1) & 1));
                    if (role_z) {
                        constexpr int HALF = ZT::TILE_BYTES / 2;
                        unsigned char* dst = land + h * HALF;
                        tma::mbar_expect_tx(&full[h], HALF);
                        if constexpr (FWD) {             // rows of the real input (HBM stream)
                            const unsigned char* src = reinterpret_cast<const unsigned char*>(a.in) + (long long)x * plane_bytes +
                                                       (long long)j * ZT::TILE_BYTES + h * HALF;
                            for (int o = 0; o < HALF; o += CHUNK)
                                tma::bulk_load_h(dst + o, src + o, HALF - o < CHUNK ? HALF - o : CHUNK, &full[h], pol_stream);
                        } else {                         // RPT/2 rows gathered from the column-tiled ring: one box
                            tma::load4_h(dst, &ring_map, &full[h], 0, 0, j * RPT + h * (RPT / 2), x % a.R, pol_keep);
                        }
                    } else {
                        constexpr int HALF = YT::TILE_BYTES / 2;
                        unsigned char* dst = land + h * HALF;
                        tma::mbar_expect_tx(&full[h], HALF);
                        if constexpr (FWD) {             // column tile j of the ring plane: one contiguous block
                            const unsigned char* src = reinterpret_cast<const unsigned char*>(a.ring) +
                                                       (long long)(x % a.R) * plane_bytes + (long long)j * YT::TILE_BYTES + h * HALF;
                            for (int o = 0; o < HALF; o += CHUNK)
                                tma::bulk_load_h(dst + o, src + o, HALF - o < CHUNK ? HALF - o : CHUNK, &full[h], pol_keep);
                        } else {                         // columns of plane x gathered from the slab layout
                            const int nb = NY / 2 / a.rows_slab;
                            for (int b = 0; b < nb; ++b) {
                                const int r0 = h * (NY / 2) + b * a.rows_slab;
                                tma::load4_h(dst + (size_t)b * a.rows_slab * YT::ROW_BYTES, &slab_map, &full[h],
                                             j * TC * W, r0 % a.L, x, r0 / a.L, pol_stream);
                            }
                        }
                    }
                }
            }
        } else if ((tid & 31) == 0) {
            // ------------------------- store thread of group my_g -------------------------
            const int my_g = (tid - NCONS) / 32 - 1;
            const unsigned long long pol_stream = tma::policy_evict_first(), pol_keep = tma::policy_evict_last();
            const unsigned char* src = work + my_g * FT::WORK_BYTES;
            int i = 0, n = 0, freed = -1;
            for (int g = rank; g < total; g += nrole, ++i) {
                if (i % NG != my_g) continue;
                const int x = g / nper, j = g - x * nper;
                tma::mbar_wait(&wdone[my_g], (unsigned)(n & 1));
                if (my_p1 && x >= a.R && x - a.R > freed) {               // ring slot must have been read out
                    tma::wait_count_bounded(&p2_loaded[x - a.R], (unsigned)n2);
                    freed = x - a.R;
                }
                if (role_z) {
                    if constexpr (FWD) {                 // RPT rows scattered into the column-tiled ring: one box
                        tma::store4_h(&ring_map, src, 0, 0, j * RPT, x % a.R, pol_keep);
                    } else {                             // rows of the real output (HBM stream)
                        unsigned char* dst = reinterpret_cast<unsigned char*>(a.out) + (long long)x * plane_bytes +
                                             (long long)j * ZT::TILE_BYTES;
                        for (int o = 0; o < ZT::TILE_BYTES; o += CHUNK)
                            tma::bulk_store_h(dst + o, src + o, ZT::TILE_BYTES - o < CHUNK ? ZT::TILE_BYTES - o : CHUNK, pol_stream);
                    }
                } else {
                    if constexpr (FWD) {                 // rows go to their slab addresses (steps 2-4 as addressing)
                        const int nb = NY / a.rows_slab;
                        for (int b = 0; b < nb; ++b) {
                            const int r0 = b * a.rows_slab;
                            tma::store4_h(&slab_map, src + (size_t)b * a.rows_slab * YT::ROW_BYTES,
                                          j * TC * W, r0 % a.L, x, r0 / a.L, pol_stream);
                        }
                    } else {                             // column tile j of the ring plane: one contiguous block
                        unsigned char* dst = reinterpret_cast<unsigned char*>(a.ring) +
                                             (long long)(x % a.R) * plane_bytes + (long long)j * YT::TILE_BYTES;
                        for (int o = 0; o < YT::TILE_BYTES; o += CHUNK)
                            tma::bulk_store_h(dst + o, src + o, YT::TILE_BYTES - o < CHUNK ? YT::TILE_BYTES - o : CHUNK, pol_keep);
                    }
                }
                tma::store_commit();
                tma::store_wait_read0();                 // the work buffer has been read out
                tma::mbar_arrive(&wfree[my_g]);
                if (my_p1) {
                    // publish at once: a deferred release would make this plane's readers depend on a LATER
                    // tile of this CTA, and with the ring's back-pressure that closes a cycle
                    tma::store_wait_all();
                    tma::fence_proxy_async_all();
                    tma::red_release_add(&p1_done[x], 1u);
                }
                ++n;
            }
            tma::store_wait_all();
        }
        return;
    }

    // ---------------- consumers: group gq takes the CTA's tiles gq, gq+NG, ... ----------------
    const int gq = tid / GROUP, gt = tid % GROUP;
    const GroupSync sync{1 + gq, GROUP};
    C* buf = reinterpret_cast<C*>(work + gq * FT::WORK_BYTES);
    const C* lnd = reinterpret_cast<const C*>(land);
    // z-tile role: thread tz of row rr
    const int tz = gt % ZCfg::S, rr = gt / ZCfg::S;
    const SmLayout<1, 0> z_dense{rr * M};
    const SmLayout<1, ZT::PADR> z_padded{rr * ZT::PITCH};
    C* scr = scratch + gq * (RPT * ZCfg::P) + rr * ZCfg::P;
    C wt = mk<T>((T)1, (T)0);                            // exp(-2 pi i t/Nz), conjugated for the inverse
    if constexpr (!C2C) {
        wt = reinterpret_cast<const C*>(a.twz)[tz];
        if constexpr (DIR > 0) wt.y = -wt.y;
    }
    const T scale = (T)a.scale;
    // y-tile role: thread ty of column cc
    const int cc = gt % TC, ty = gt / TC;
    const SmLayout<TC, 0> y_dense{cc};
    const SmLayout<TC, YT::PADR> y_padded{cc};

    int i = 0, n = 0;                                    // CTA tile index, group-local tile index
    for (int g = rank; g < total; g += nrole, ++i) {
        if (i % NG != gq) continue;
        const int x = g / nper;
        while (*turn < i) { }
        const unsigned par = (unsigned)(i & 1);
        // the group's store thread has read the previous output tile out of the work buffer
        auto work_free = [&]() { if (n > 0) tma::mbar_wait(&wfree[gq], (unsigned)((n - 1) & 1)); };
        if (role_z) {
            constexpr int P = ZCfg::P;
            C v[P];
            const int h = gt / (GROUP / 2);              // rows [0, RPT/2) land in half 0
            tma::mbar_wait(&full[h], par);
            read_own<ZCfg, T>(v, lnd, tz, z_dense);
            __syncwarp();
            if ((tid & 31) == 0) tma::mbar_arrive(&empty[h]);
            if (gt == 0) {
                tma::mbar_wait(&full[1], par);           // both phases of tile i are over: the next group may wait
                *turn = i + 1;
                if (!my_p1) tma::red_release_add(&p2_loaded[x], 1u);      // the ring tile has been read
            }
            if constexpr (DIR > 0 && !C2C) {
                if (tz == 0) {
#pragma unroll
                    for (int m = 0; m < P; ++m) scr[m] = v[m];
                }
                __syncwarp();
                hermitian_step<ZCfg, true, T>(v, wt, tz, scr);
                __syncwarp();
            }
            if constexpr (ZCfg::NST > 1) fft_stages<ZCfg, 0, DIR, T>(v, buf, tw_s, tz, z_padded, sync, work_free);
            else { fft_stages<ZCfg, 0, DIR, T>(v, buf, tw_s, tz, z_padded, sync); work_free(); }
            if constexpr (DIR < 0 && !C2C) {
                if (tz == 0) {
#pragma unroll
                    for (int m = 0; m < P; ++m) scr[m] = v[m];
                }
                __syncwarp();
                hermitian_step<ZCfg, false, T>(v, wt, tz, scr);
                __syncwarp();
            } else if constexpr (DIR > 0) {
#pragma unroll
                for (int m = 0; m < P; ++m) v[m] = mk<T>(v[m].x * scale, v[m].y * scale);
            }
            if constexpr (ZCfg::NST > 1) sync();         // all exchange reads done: the buffer becomes the output tile
            write_own<ZCfg, T>(v, buf, tz, z_dense);
        } else {
            constexpr int P = YCfg::P;
            C v[P];
            tma::mbar_wait(&full[0], par);               // rows [0, Ny/2): elements t + m*S, m < P/2
            read_own_range<YCfg, 0, P / 2, T>(v, lnd, ty, y_dense);
            __syncwarp();
            if ((tid & 31) == 0) tma::mbar_arrive(&empty[0]);
            tma::mbar_wait(&full[1], par);
            read_own_range<YCfg, P / 2, P, T>(v, lnd, ty, y_dense);
            __syncwarp();
            if ((tid & 31) == 0) tma::mbar_arrive(&empty[1]);
            if (gt == 0) {
                *turn = i + 1;
                if (!my_p1) tma::red_release_add(&p2_loaded[x], 1u);      // the ring tile has been read
            }
            if constexpr (YCfg::NST > 1) fft_stages<YCfg, 0, DIR, T>(v, buf, tw_s, ty, y_padded, sync, work_free);
            else { fft_stages<YCfg, 0, DIR, T>(v, buf, tw_s, ty, y_padded, sync); work_free(); }
            if constexpr (YCfg::NST > 1) sync();
            write_own<YCfg, T>(v, buf, ty, y_dense);
        }
        tma::fence_proxy_async();
        __syncwarp();
        if ((tid & 31) == 0) tma::mbar_arrive(&wdone[gq]);
        ++n;
    }
}

}  // namespace fft3d
