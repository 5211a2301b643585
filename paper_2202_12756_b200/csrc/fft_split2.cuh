// fft_split2.cuh -- Y passes (F2, I2; paper step 1 y half + steps 2-4, P:69-76 / P:86) for lengths whose
// [N rows][TC columns] tile is too large for more than ONE ring stage (N = 2048 fp32: 128 KiB), so that
// load, transform and store take turns (3.5 TB/s).
//
// One decimation-in-time step is taken OUT of the tile: the even rows and the odd rows of a tile are two
// independent N/2-point transforms E and O, each a half tile of 64 KiB that moves through a 3-slot ring
// like any other tile; when the second one is done the two are combined in place, element by element,
//     X[k] = E[k] + w^k O[k],   X[k + N/2] = E[k] - w^k O[k],   w = exp(-+2 pi i / N),
// after which the slot that held E holds output rows [0, N/2) and the slot that held O rows [N/2, N).
// The loads of the next tile's even half overlap the transform of this tile's odd half, and so on.
// Each thread combines exactly the elements it wrote itself (t + m*S), so the combine needs no barrier;
// w^(t + m S) = w^t * exp(-+2 pi i m / (2P)): one per-thread value times compile-time constants.
//
// Even / odd rows are addressed by tensor maps with a doubled row stride (built per call on the host).
#pragma once
#include "fft_kernels.cuh"

namespace fft3d {

// X[k] = E[k] + w^k O[k] -> e, X[k+H] = E[k] - w^k O[k] -> o, for the thread's own elements k = t + m*S
// (O in registers, E in its slot's dense layout)
template <class HCfg, int DIR, typename T, class Lay, int MM = 0>
__device__ __forceinline__ void combine_halves(cx<T> (&v)[HCfg::P], cx<T>* __restrict__ e, cx<T>* __restrict__ o,
                                               cx<T> wt, int t, const Lay& lay) {
    if constexpr (MM < HCfg::P) {
        constexpr int P = HCfg::P, S = HCfg::S;
        const int idx = lay.at(t + MM * S);
        const cx<T> wo = cmul(mul_root<MM, 2 * P, DIR, T>(wt), v[MM]);
        const cx<T> ev = e[idx];
        e[idx] = cadd(ev, wo);
        o[idx] = csub(ev, wo);
        combine_halves<HCfg, DIR, T, Lay, MM + 1>(v, e, o, wt, t, lay);
    }
}

// HCfg: the N/2-point transform.  PASS: TMA_Y_FWD (natural -> slab) or TMA_Y_INV (slab -> natural).
template <class HCfg, int TC, int PASS, typename T, int NSTAGE>
__global__ void __launch_bounds__(HCfg::S * TC + 32, 1)
fft_y_split2_kernel(const __grid_constant__ TensorMapBlob in_even, const __grid_constant__ TensorMapBlob in_odd,
                    const __grid_constant__ TensorMapBlob out_map, const TmaArgs a) {
    using C = cx<T>;
    using TT = TmaTile<HCfg, TC, T, false>;
    constexpr int P = HCfg::P, W = TT::W, NCONS = TT::NCONS, H = HCfg::N;   // H = N/2 rows per half
    constexpr int DIR = (PASS == TMA_Y_FWD) ? -1 : +1;
    static_assert(PASS == TMA_Y_FWD || PASS == TMA_Y_INV, "Y passes only");
    static_assert(NSTAGE >= 3, "a pair of half tiles plus one in flight");
    extern __shared__ __align__(1024) unsigned char smem_dyn[];
    C* tw = reinterpret_cast<C*>(smem_dyn);
    unsigned char* stages = smem_dyn + TT::TW_BYTES;
    unsigned long long* full = reinterpret_cast<unsigned long long*>(stages + NSTAGE * TT::STAGE_BYTES);
    unsigned long long* done = full + NSTAGE;

    const int tid = threadIdx.x;
    const bool is_producer = tid >= NCONS;
    if (tid == NCONS) {
        for (int s = 0; s < NSTAGE; ++s) { tma::mbar_init(&full[s], 1); tma::mbar_init(&done[s], NCONS / 32); }
        tma::fence_mbar_init();
    }
    if (!is_producer) load_twiddles<DIR, T>(tw, reinterpret_cast<const C*>(a.tw), HCfg::TWN, tid, NCONS);
    __syncthreads();

    const long long first = blockIdx.x, stride = gridDim.x;
    const long long n_tiles = first < a.ntiles ? (a.ntiles - first + stride - 1) / stride : 0;
    const long long n_items = 2 * n_tiles;               // item i = (tile i/2, half i&1)
    const int Lh = a.L / 2;                              // half rows per virtual slab

    if (is_producer) {
        if (tid != NCONS) return;
        auto issue_load = [=, &in_even, &in_odd](long long i) {
            const long long t_id = first + (i >> 1) * stride;
            const int h = (int)(i & 1), s = (int)(i % NSTAGE);
            const int tz = (int)(t_id % a.ntz), x = (int)(t_id / a.ntz);
            unsigned char* dst = stages + s * TT::STAGE_BYTES;
            const TensorMapBlob* map = h ? &in_odd : &in_even;
            const int nb = H / a.in_rows;
            tma::mbar_expect_tx(&full[s], TT::TILE_BYTES);
            for (int b = 0; b < nb; ++b) {
                void* d = dst + (size_t)b * a.in_rows * TT::ROW_BYTES;
                const int r0 = b * a.in_rows;                    // index among the even (odd) rows
                if constexpr (PASS == TMA_Y_FWD) tma::load3(d, map, &full[s], tz * TC * W, r0, x);
                else tma::load4(d, map, &full[s], tz * TC * W, r0 % Lh, x, r0 / Lh);
            }
        };
        // output rows [h*H, (h+1)*H) of the tile sit in the slot of its half h
        auto issue_store = [=, &out_map](long long i) {
            const long long t_id = first + (i >> 1) * stride;
            const int h = (int)(i & 1), s = (int)(i % NSTAGE);
            const int tz = (int)(t_id % a.ntz), x = (int)(t_id / a.ntz);
            const unsigned char* src = stages + s * TT::STAGE_BYTES;
            const int nb = H / a.out_rows;
            for (int b = 0; b < nb; ++b) {
                const void* d = src + (size_t)b * a.out_rows * TT::ROW_BYTES;
                const int r0 = h * H + b * a.out_rows;
                if constexpr (PASS == TMA_Y_FWD) tma::store4(&out_map, d, tz * TC * W, r0 % a.L, x, r0 / a.L);
                else tma::store3(&out_map, d, tz * TC * W, r0, x);
            }
        };
        long long stored_pairs = 0;
        auto ensure_stored = [&](long long j) {                  // item j's slot is reusable after its pair is out
            const long long pr = j >> 1;
            if (pr < stored_pairs) return;
            for (long long k = 2 * pr; k < 2 * pr + 2; ++k)
                tma::mbar_wait(&done[k % NSTAGE], (unsigned)((k / NSTAGE) & 1));
            issue_store(2 * pr);
            issue_store(2 * pr + 1);
            tma::store_commit();
            tma::store_wait_read0();
            stored_pairs = pr + 1;
        };
        for (long long i = 0; i < n_items; ++i) {
            if (i >= NSTAGE) ensure_stored(i - NSTAGE);
            issue_load(i);
        }
        for (long long pr = stored_pairs; pr < n_tiles; ++pr) ensure_stored(2 * pr);
        tma::store_wait_all();
        return;
    }

    // ---------------- consumers ----------------
    const int c = tid % TC, t = tid / TC;
    const SmLayout<TC, 0> dense{c};
    const SmLayout<TC, TT::PADR> padded{c};
    const NamedSync<1, NCONS> sync{};
    // w^t = exp(DIR 2 pi i t / N), N = 2H, in double once per thread (no fast-math intrinsics)
    double ws, wc;
    sincospi((double)DIR * (double)t / (double)H, &ws, &wc);
    const C wt = mk<T>((T)wc, (T)ws);
    for (long long i = 0; i < n_items; ++i) {
        const int s = (int)(i % NSTAGE);
        C* buf = reinterpret_cast<C*>(stages + s * TT::STAGE_BYTES);
        tma::mbar_wait(&full[s], (unsigned)((i / NSTAGE) & 1));
        C v[P];
        read_own<HCfg, T>(v, buf, t, dense);
        if constexpr (HCfg::NST > 1) sync();
        fft_stages<HCfg, 0, DIR, T>(v, buf, tw, t, padded, sync);
        if constexpr (HCfg::NST > 1) sync();                     // all exchange reads done
        if ((i & 1) == 0) {
            write_own<HCfg, T>(v, buf, t, dense);                // E stays in its slot until O is there
        } else {
            C* ebuf = reinterpret_cast<C*>(stages + (int)((i - 1) % NSTAGE) * TT::STAGE_BYTES);
            combine_halves<HCfg, DIR, T>(v, ebuf, buf, wt, t, dense);
            tma::fence_proxy_async();
            __syncwarp();
            if ((tid & 31) == 0) { tma::mbar_arrive(&done[(i - 1) % NSTAGE]); tma::mbar_arrive(&done[s]); }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// The same for the X passes (F3, I1; paper step 5, P:77 / P:86) with the shifted windows of odd rows
// (fft_kernels.cuh, ODDFIX): used where a whole tile with its TC+2 landing columns leaves room for one
// ring stage only (Nx = 1536 fp32: 120 KiB) but a half tile for three (60 KiB).
//   loads: ld_even / ld_odd = the even / odd x rows of the loading side, plain windows (TC columns);
//          ldw_even / ldw_odd = the same with TC+2 columns (windows of odd-l rows);  store: the whole array.
// ---------------------------------------------------------------------------------------------
template <class HCfg, int TC, int PASS, typename T, int NSTAGE>
__global__ void __launch_bounds__(HCfg::S * TC + 32, 1)
fft_x_split2_kernel(const __grid_constant__ TensorMapBlob ld_even, const __grid_constant__ TensorMapBlob ld_odd,
                    const __grid_constant__ TensorMapBlob ldw_even, const __grid_constant__ TensorMapBlob ldw_odd,
                    const __grid_constant__ TensorMapBlob out_map, const TmaArgs a) {
    using C = cx<T>;
    using TT = TmaTile<HCfg, TC, T, true>;
    constexpr int P = HCfg::P, S = HCfg::S, W = TT::W, NCONS = TT::NCONS, H = HCfg::N;
    constexpr int DIR = (PASS == TMA_X_FWD) ? -1 : +1;
    static_assert(PASS == TMA_X_FWD || PASS == TMA_X_INV, "X passes only");
    static_assert(NSTAGE >= 3, "a pair of half tiles plus one in flight");
    extern __shared__ __align__(1024) unsigned char smem_dyn[];
    C* tw = reinterpret_cast<C*>(smem_dyn);
    unsigned char* stages = smem_dyn + TT::TW_BYTES;
    unsigned long long* full = reinterpret_cast<unsigned long long*>(stages + NSTAGE * TT::STAGE_BYTES);
    unsigned long long* done = full + NSTAGE;

    const int tid = threadIdx.x;
    const bool is_producer = tid >= NCONS;
    if (tid == NCONS) {
        for (int s = 0; s < NSTAGE; ++s) { tma::mbar_init(&full[s], 1); tma::mbar_init(&done[s], NCONS / 32); }
        tma::fence_mbar_init();
    }
    if (!is_producer) load_twiddles<DIR, T>(tw, reinterpret_cast<const C*>(a.tw), HCfg::TWN, tid, NCONS);
    __syncthreads();

    const long long first = blockIdx.x, stride = gridDim.x;
    const long long n_tiles = first < a.ntiles ? (a.ntiles - first + stride - 1) / stride : 0;
    const long long n_items = 2 * n_tiles;

    if (is_producer) {
        if (tid != NCONS) return;
        auto issue_load = [=, &ld_even, &ld_odd, &ldw_even, &ldw_odd](long long i) {
            const XTile xt = decode_xtile<PASS, true>(first + (i >> 1) * stride, a, TC);
            const int h = (int)(i & 1), s = (int)(i % NSTAGE);
            unsigned char* dst = stages + s * TT::STAGE_BYTES;
            const int rowb = xt.odd ? TT::ROW_BYTES_WIDE : TT::ROW_BYTES;
            const TensorMapBlob* map = xt.odd ? (h ? &ldw_odd : &ldw_even) : (h ? &ld_odd : &ld_even);
            const int nb = H / a.in_rows;
            tma::mbar_expect_tx(&full[s], (unsigned)(H * rowb));
            for (int b = 0; b < nb; ++b) {
                void* d = dst + (size_t)b * a.in_rows * rowb;
                const int r0 = b * a.in_rows;                    // index among the even (odd) x rows
                if constexpr (PASS == TMA_X_FWD)
                    tma::load4(d, map, &full[s], (xt.k0 - xt.odd) * W, xt.l, r0, xt.q);
                else
                    tma::load3(d, map, &full[s], (xt.l * a.Mp1 + xt.w * TC - xt.odd) * W, r0, xt.q);
            }
        };
        const unsigned long long pol_keep = tma::make_policy_evict_last();   // see fft_strided_tma_kernel
        auto issue_store = [=, &out_map](long long i) {
            const XTile xt = decode_xtile<PASS, true>(first + (i >> 1) * stride, a, TC);
            if (xt.thin) return;                                 // stored by the consumers
            const int h = (int)(i & 1), s = (int)(i % NSTAGE);
            const unsigned char* src = stages + s * TT::STAGE_BYTES;
            const int nb = H / a.out_rows;
            for (int b = 0; b < nb; ++b) {
                const void* d = src + (size_t)b * a.out_rows * TT::ROW_BYTES;
                const int r0 = h * H + b * a.out_rows;
                if constexpr (PASS == TMA_X_FWD)
                    tma::store3_hint(&out_map, d, (xt.l * a.Mp1 + xt.k0) * W, r0, xt.q, pol_keep);
                else
                    tma::store4(&out_map, d, xt.w * TC * W, xt.l, r0, xt.q);
            }
        };
        long long stored_pairs = 0;
        auto ensure_stored = [&](long long j) {
            const long long pr = j >> 1;
            if (pr < stored_pairs) return;
            for (long long k = 2 * pr; k < 2 * pr + 2; ++k)
                tma::mbar_wait(&done[k % NSTAGE], (unsigned)((k / NSTAGE) & 1));
            issue_store(2 * pr);
            issue_store(2 * pr + 1);
            tma::store_commit();
            tma::store_wait_read0();
            stored_pairs = pr + 1;
        };
        for (long long i = 0; i < n_items; ++i) {
            if (i >= NSTAGE) ensure_stored(i - NSTAGE);
            issue_load(i);
        }
        for (long long pr = stored_pairs; pr < n_tiles; ++pr) ensure_stored(2 * pr);
        tma::store_wait_all();
        return;
    }

    // ---------------- consumers ----------------
    const int c = tid % TC, t = tid / TC;
    const SmLayout<TC, 0> dense{c};
    const SmLayout<TC + 2, 0> dense_wide{c + 1};
    const SmLayout<TC, TT::PADR> padded{c};
    const NamedSync<1, NCONS> sync{};
    double ws, wc;
    sincospi((double)DIR * (double)t / (double)H, &ws, &wc);
    const C wt = mk<T>((T)wc, (T)ws);
    for (long long i = 0; i < n_items; ++i) {
        const XTile xt = decode_xtile<PASS, true>(first + (i >> 1) * stride, a, TC);
        const int s = (int)(i % NSTAGE);
        C* buf = reinterpret_cast<C*>(stages + s * TT::STAGE_BYTES);
        tma::mbar_wait(&full[s], (unsigned)((i / NSTAGE) & 1));
        C v[P];
        if (xt.odd) read_own<HCfg, T>(v, buf, t, dense_wide);
        else read_own<HCfg, T>(v, buf, t, dense);
        if constexpr (HCfg::NST > 1) sync();
        fft_stages<HCfg, 0, DIR, T>(v, buf, tw, t, padded, sync);
        if constexpr (HCfg::NST > 1) sync();
        if ((i & 1) == 0) {
            write_own<HCfg, T>(v, buf, t, dense);
        } else {
            C* ebuf = reinterpret_cast<C*>(stages + (int)((i - 1) % NSTAGE) * TT::STAGE_BYTES);
            combine_halves<HCfg, DIR, T>(v, ebuf, buf, wt, t, dense);
            if (PASS == TMA_X_FWD && xt.thin) {
                // thin tile: only column M-1 (thread column 0) is real; plain stores to the user's rows
                __syncwarp();
                if (c >= xt.c_lo && c < xt.c_hi) {
                    const long long rstride = (long long)a.L * a.Mp1;
                    C* p = reinterpret_cast<C*>(a.user_out) +
                           (((long long)xt.q * a.Nx * a.L + xt.l) * a.Mp1 + (xt.k0 + c));
#pragma unroll
                    for (int m = 0; m < P; ++m) {
                        const int k = t + m * S;
                        p[(long long)k * rstride] = ebuf[dense.at(k)];
                        p[(long long)(k + H) * rstride] = buf[dense.at(k)];
                    }
                }
            }
            tma::fence_proxy_async();
            __syncwarp();
            if ((tid & 31) == 0) { tma::mbar_arrive(&done[(i - 1) % NSTAGE]); tma::mbar_arrive(&done[s]); }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// Two decimation-in-time steps taken out of the tile: the X passes of Nx = 2048 fp32, whose odd-row half
// tiles land 80 KiB (three slots do not fit) but whose QUARTER tiles land 40 KiB (five slots do).  Rows
// x = 4k + m, m = 0..3, are four independent Nx/4-point transforms Q_m; when the fourth is done
//     X[k + j Nx/4] = sum_m (-+i)^(j m) w^(m k) Q_m[k],   w = exp(-+2 pi i / Nx),
// element by element (a radix-4 butterfly on the thread's own elements, no barrier), and the four slots hold
// output rows [j Nx/4, (j+1) Nx/4).  Loads: ld[wide][m] = rows x = m (mod 4) of the loading side, plain / wide.
// ---------------------------------------------------------------------------------------------
struct Split4Maps { TensorMapBlob ld[2][4]; };

template <class QCfg, int DIR, typename T, class Lay, int MM = 0>
__device__ __forceinline__ void combine_quarters(cx<T> (&v)[QCfg::P], cx<T>* q0, cx<T>* q1, cx<T>* q2, cx<T>* q3,
                                                 const cx<T> (&wt)[3], int t, const Lay& lay, cx<T>* thin_p, long long rstride,
                                                 bool thin) {
    if constexpr (MM < QCfg::P) {
        constexpr int P = QCfg::P, S = QCfg::S, H4 = QCfg::N;
        const int k = t + MM * S, idx = lay.at(k);
        cx<T> a[4];
        a[0] = q0[idx];
        a[1] = cmul(mul_root<MM, 4 * P, DIR, T>(wt[0]), q1[idx]);
        a[2] = cmul(mul_root<2 * MM, 4 * P, DIR, T>(wt[1]), q2[idx]);
        a[3] = cmul(mul_root<3 * MM, 4 * P, DIR, T>(wt[2]), v[MM]);
        dft<4, DIR, T>(a);
        if (thin) {
            if (thin_p != nullptr) {
#pragma unroll
                for (int j = 0; j < 4; ++j) thin_p[(long long)(k + j * H4) * rstride] = a[j];
            }
        } else {
            q0[idx] = a[0]; q1[idx] = a[1]; q2[idx] = a[2]; q3[idx] = a[3];
        }
        combine_quarters<QCfg, DIR, T, Lay, MM + 1>(v, q0, q1, q2, q3, wt, t, lay, thin_p, rstride, thin);
    }
}

template <class QCfg, int TC, int PASS, typename T, int NSTAGE>
__global__ void __launch_bounds__(QCfg::S * TC + 32, 1)
fft_x_split4_kernel(const __grid_constant__ Split4Maps maps, const __grid_constant__ TensorMapBlob out_map, const TmaArgs a) {
    using C = cx<T>;
    using TT = TmaTile<QCfg, TC, T, true>;
    constexpr int P = QCfg::P, W = TT::W, NCONS = TT::NCONS, H4 = QCfg::N;
    constexpr int DIR = (PASS == TMA_X_FWD) ? -1 : +1;
    static_assert(PASS == TMA_X_FWD || PASS == TMA_X_INV, "X passes only");
    static_assert(NSTAGE >= 5, "four quarter tiles plus one in flight");
    extern __shared__ __align__(1024) unsigned char smem_dyn[];
    C* tw = reinterpret_cast<C*>(smem_dyn);
    unsigned char* stages = smem_dyn + TT::TW_BYTES;
    unsigned long long* full = reinterpret_cast<unsigned long long*>(stages + NSTAGE * TT::STAGE_BYTES);
    unsigned long long* done = full + NSTAGE;

    const int tid = threadIdx.x;
    const bool is_producer = tid >= NCONS;
    if (tid == NCONS) {
        for (int s = 0; s < NSTAGE; ++s) { tma::mbar_init(&full[s], 1); tma::mbar_init(&done[s], NCONS / 32); }
        tma::fence_mbar_init();
    }
    if (!is_producer) load_twiddles<DIR, T>(tw, reinterpret_cast<const C*>(a.tw), QCfg::TWN, tid, NCONS);
    __syncthreads();

    const long long first = blockIdx.x, stride = gridDim.x;
    const long long n_tiles = first < a.ntiles ? (a.ntiles - first + stride - 1) / stride : 0;
    const long long n_items = 4 * n_tiles;               // item i = (tile i/4, quarter i&3)

    if (is_producer) {
        if (tid != NCONS) return;
        const unsigned long long pol_keep = tma::make_policy_evict_last();
        auto issue_load = [=, &maps](long long i) {
            const XTile xt = decode_xtile<PASS, true>(first + (i >> 2) * stride, a, TC);
            const int m = (int)(i & 3), s = (int)(i % NSTAGE);
            unsigned char* dst = stages + s * TT::STAGE_BYTES;
            const int rowb = xt.odd ? TT::ROW_BYTES_WIDE : TT::ROW_BYTES;
            const TensorMapBlob* map = &maps.ld[xt.odd][m];
            const int nb = H4 / a.in_rows;
            tma::mbar_expect_tx(&full[s], (unsigned)(H4 * rowb));
            for (int b = 0; b < nb; ++b) {
                void* d = dst + (size_t)b * a.in_rows * rowb;
                const int r0 = b * a.in_rows;
                if constexpr (PASS == TMA_X_FWD)
                    tma::load4(d, map, &full[s], (xt.k0 - xt.odd) * W, xt.l, r0, xt.q);
                else
                    tma::load3(d, map, &full[s], (xt.l * a.Mp1 + xt.w * TC - xt.odd) * W, r0, xt.q);
            }
        };
        auto issue_store = [=, &out_map](long long i) {
            const XTile xt = decode_xtile<PASS, true>(first + (i >> 2) * stride, a, TC);
            if (xt.thin) return;
            const int j = (int)(i & 3), s = (int)(i % NSTAGE);
            const unsigned char* src = stages + s * TT::STAGE_BYTES;
            const int nb = H4 / a.out_rows;
            for (int b = 0; b < nb; ++b) {
                const void* d = src + (size_t)b * a.out_rows * TT::ROW_BYTES;
                const int r0 = j * H4 + b * a.out_rows;
                if constexpr (PASS == TMA_X_FWD)
                    tma::store3_hint(&out_map, d, (xt.l * a.Mp1 + xt.k0) * W, r0, xt.q, pol_keep);
                else
                    tma::store4(&out_map, d, xt.w * TC * W, xt.l, r0, xt.q);
            }
        };
        long long stored_tiles = 0;
        auto ensure_stored = [&](long long j) {
            const long long tl = j >> 2;
            if (tl < stored_tiles) return;
            for (long long k = 4 * tl; k < 4 * tl + 4; ++k)
                tma::mbar_wait(&done[k % NSTAGE], (unsigned)((k / NSTAGE) & 1));
            for (long long k = 4 * tl; k < 4 * tl + 4; ++k) issue_store(k);
            tma::store_commit();
            tma::store_wait_read0();
            stored_tiles = tl + 1;
        };
        for (long long i = 0; i < n_items; ++i) {
            if (i >= NSTAGE) ensure_stored(i - NSTAGE);
            issue_load(i);
        }
        for (long long tl = stored_tiles; tl < n_tiles; ++tl) ensure_stored(4 * tl);
        tma::store_wait_all();
        return;
    }

    // ---------------- consumers ----------------
    const int c = tid % TC, t = tid / TC;
    const SmLayout<TC, 0> dense{c};
    const SmLayout<TC + 2, 0> dense_wide{c + 1};
    const SmLayout<TC, TT::PADR> padded{c};
    const NamedSync<1, NCONS> sync{};
    C wt[3];                                             // w^(j t), j = 1..3, w = exp(DIR 2 pi i / N), N = 4 H4
#pragma unroll
    for (int j = 1; j <= 3; ++j) {
        double ws, wc;
        sincospi((double)DIR * (double)(j * t) / (double)(2 * H4), &ws, &wc);
        wt[j - 1] = mk<T>((T)wc, (T)ws);
    }
    for (long long i = 0; i < n_items; ++i) {
        const XTile xt = decode_xtile<PASS, true>(first + (i >> 2) * stride, a, TC);
        const int s = (int)(i % NSTAGE);
        C* buf = reinterpret_cast<C*>(stages + s * TT::STAGE_BYTES);
        tma::mbar_wait(&full[s], (unsigned)((i / NSTAGE) & 1));
        C v[P];
        if (xt.odd) read_own<QCfg, T>(v, buf, t, dense_wide);
        else read_own<QCfg, T>(v, buf, t, dense);
        if constexpr (QCfg::NST > 1) sync();
        fft_stages<QCfg, 0, DIR, T>(v, buf, tw, t, padded, sync);
        if constexpr (QCfg::NST > 1) sync();
        if ((i & 3) != 3) {
            write_own<QCfg, T>(v, buf, t, dense);
        } else {
            C* q0 = reinterpret_cast<C*>(stages + (int)((i - 3) % NSTAGE) * TT::STAGE_BYTES);
            C* q1 = reinterpret_cast<C*>(stages + (int)((i - 2) % NSTAGE) * TT::STAGE_BYTES);
            C* q2 = reinterpret_cast<C*>(stages + (int)((i - 1) % NSTAGE) * TT::STAGE_BYTES);
            const bool thin = PASS == TMA_X_FWD && xt.thin;
            const long long rstride = (long long)a.L * a.Mp1;
            C* thin_p = nullptr;
            if (thin && c >= xt.c_lo && c < xt.c_hi)
                thin_p = reinterpret_cast<C*>(a.user_out) + (((long long)xt.q * a.Nx * a.L + xt.l) * a.Mp1 + (xt.k0 + c));
            combine_quarters<QCfg, DIR, T>(v, q0, q1, q2, buf, wt, t, dense, thin_p, rstride, thin);
            tma::fence_proxy_async();
            __syncwarp();
            if ((tid & 31) == 0) {
#pragma unroll
                for (int j = 0; j < 4; ++j) tma::mbar_arrive(&done[(i - 3 + j) % NSTAGE]);
            }
        }
    }
}

}  // namespace fft3d
