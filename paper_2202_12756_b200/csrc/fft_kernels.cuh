// fft_kernels.cuh -- the full-array passes of the slab 3D FFT:
//
//   fft_z_r2c_kernel        pass F1: rows of Nz reals -> Nz/2 packed complex (paper step 1, z half)
//   fft_z_c2r_kernel        pass I3: the mirror image, with the 1/(NxNyNz) normalisation fused
//   fft_strided_tma_kernel  passes F2, F3, I1, I2 on sm_100a: C2C FFT down a strided axis on a
//                           [N rows][TC cols] tile, tiles streamed by TMA through a shared-memory ring
//   fft_strided_kernel      the same passes with plain loads/stores (any extent / alignment; also the
//                           ablation baseline, fft3d_set_variant(plan, 1))
//
// In the y passes the row index is split as row = q*L + l on one side, which is how the paper's local
// transpose + all-to-all + chunk transpose (steps 2-4) are folded into the pass as pure
// addressing.
//
// "Packed" complex rows: the z pass keeps Nz/2 columns; column 0 holds (X[0], X[Nz/2]) -- both
// real after an R2C -- as one complex number.  The strided passes are linear, so column 0 then
// carries A + iB with A, B the transforms of two real planes; fft3d_fixup.cu separates them.
#pragma once
#include <cstdint>

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
    long long out_cs;            // element stride between output columns (0 means 1)
};

struct ZArgs {
    const void* in;
    void* out;
    const void* tw;              // stage twiddles for the M = Nz/2 point FFT
    const void* twz;             // exp(-2 pi i k / Nz), k < M
    long long nrows;
    double scale;                // C2R only: 1/(Nx Ny Nz)
    long long in_pitch, out_pitch;   // complex elements between consecutive rows (0 = M, dense); M+1 for the padded
                                     // in-place layout (rows of Nz+2 reals), where in == out is allowed
};

// row padding of shared-memory tiles: one extra row every PADR rows (0 = none)
template <class Cfg, int ROW_BYTES>
struct TilePad {
    static constexpr int r0 = Cfg::radix(0);
    static constexpr int PADR = (ROW_BYTES < 128 && Cfg::NST > 1 && r0 % 4 == 0) ? r0 : 0;
    static constexpr int ROWS = Cfg::N + (PADR ? Cfg::N / PADR : 0);
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

// Global -> register load of one tile (thread (t, c) owns rows t + m*S of column c).
template <class Cfg, int TC, bool IN_SLAB, typename T>
__device__ __forceinline__ void strided_load_tile(cx<T> (&v)[Cfg::P], const StridedArgs& a, long long tid,
                                                  int t, int c, float invL) {
    using C = cx<T>;
    constexpr int P = Cfg::P, S = Cfg::S;
    const int tz = (int)(tid % a.ntz);
    const long long aa = tid / a.ntz;
    const long long a_hi = aa / a.a_lo, a_l = aa % a.a_lo;
    const int col = tz * TC + c;
    const bool ok = col < a.ncols;
    const C* in = reinterpret_cast<const C*>(a.in) + (a_hi * a.in_hi + a_l * a.in_lo + col);
    long long in_rl = a.in_rl;
    if (a.col0 != nullptr && col == 0) {      // packed column 0 comes from the side buffer
        in = reinterpret_cast<const C*>(a.col0) + (a_hi * a.c0_hi + a_l * a.c0_lo);
        in_rl = a.c0_rl;
    }
#pragma unroll
    for (int m = 0; m < P; ++m) {
        const long long off = row_offset<IN_SLAB>(t + m * S, a.L, invL, a.in_rq, in_rl);
        v[m] = ok ? in[off] : mk<T>((T)0, (T)0);
    }
}

// PREFETCH: keep the next tile's loads in flight (in a second register set) while the current
// tile is transformed -- the persistent CTA never waits on an empty memory pipeline.
template <class Cfg, int TC, int DIR, bool IN_SLAB, bool OUT_SLAB, typename T, int MINB, bool PREFETCH>
__global__ void __launch_bounds__(Cfg::S * TC, MINB) fft_strided_kernel(const StridedArgs a) {
    using C = cx<T>;
    constexpr int P = Cfg::P, S = Cfg::S;
    using Pad = TilePad<Cfg, TC * (int)sizeof(C)>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C* tw = reinterpret_cast<C*>(smem_raw);
    C* tile = tw + ((Cfg::TWN + 1) & ~1);
    load_twiddles<DIR, T>(tw, reinterpret_cast<const C*>(a.tw), Cfg::TWN, threadIdx.x, blockDim.x);

    const int c = threadIdx.x % TC, t = threadIdx.x / TC;
    const SmLayout<TC, Pad::PADR> lay{c};
    const float invL = 1.0f / (float)a.L;

    C vn[P];
    if constexpr (PREFETCH) {
        if ((long long)blockIdx.x < a.ntiles) strided_load_tile<Cfg, TC, IN_SLAB, T>(vn, a, blockIdx.x, t, c, invL);
    }
    for (long long tid = blockIdx.x; tid < a.ntiles; tid += gridDim.x) {
        C v[P];
        if constexpr (PREFETCH) {
#pragma unroll
            for (int m = 0; m < P; ++m) v[m] = vn[m];
            if (tid + gridDim.x < a.ntiles)
                strided_load_tile<Cfg, TC, IN_SLAB, T>(vn, a, tid + gridDim.x, t, c, invL);
        } else {
            strided_load_tile<Cfg, TC, IN_SLAB, T>(v, a, tid, t, c, invL);
        }
        const int tz = (int)(tid % a.ntz);
        const long long aa = tid / a.ntz;
        const long long a_hi = aa / a.a_lo, a_l = aa % a.a_lo;
        const int col = tz * TC + c;
        const bool ok = col < a.ncols;
        C* out = reinterpret_cast<C*>(a.out) + (a_hi * a.out_hi + a_l * a.out_lo + (a.out_cs ? col * a.out_cs : col));
        if constexpr (Cfg::NST > 1) __syncthreads();   // twiddles loaded / previous tile fully read
        fft_stages<Cfg, 0, DIR, T>(v, tile, tw, t, lay, CtaSync{});
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
// TMA-pipelined strided pass (sm_100a): one persistent CTA per SM, a producer warp and S*TC
// consumer threads.  The producer streams tiles into an NSTAGE-deep shared-memory ring with
// cp.async.bulk.tensor (no per-thread address arithmetic, loads run tiles ahead); the consumers
// transform a tile IN PLACE in its ring slot (dense -> padded exchange layout -> dense) and hand
// it back; the producer writes it out with a bulk tensor store and refills the slot.
//
// Tensor maps are built per call on the host (fft3d_plan.cu) in units of 8-byte words
// (W = sizeof(complex)/8 words per element).  Coordinates of box b (rows r0 = b*rows ..) of a tile:
//   Y passes (F2, I2): tile = (x, tz);   natural side  (tz*TC, r0, x)
//                                         slab side     (tz*TC, r0 % L, x, r0 / L)
//   X passes (F3, I1): tile = (q, l, w);  packed side   (w*TC, l, r0, q)
//                                         user side, rows of one (q,x) flattened to L*(M+1):
//                                                       (l*(M+1) + w*TC, r0, q)
// ---------------------------------------------------------------------------------------------
enum { TMA_Y_FWD = 0, TMA_Y_INV = 1, TMA_X_FWD = 2, TMA_X_INV = 3 };

struct TmaArgs {
    const void* tw;          // forward stage twiddles
    void* user_out;          // X_FWD with ODDFIX: the caller's spectrum (thin tiles store directly)
    long long ntiles;
    int ntz;                 // column tiles per row
    int L;                   // rows per virtual slab
    int Nx;
    int Mp1;                 // M + 1 (pitch of the user spectrum)
    int in_rows, out_rows;   // rows per TMA box on each side
    int cls4;                // X_FWD, fp32: four row classes l % 4 (every user-side window on a 32-byte sector)
};

namespace tma {
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned long long* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "WAIT_LOOP:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra.uni WAIT_DONE;\n\t"
        "bra.uni WAIT_LOOP;\n\t"
        "WAIT_DONE:\n\t}" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void fence_mbar_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void load3(void* dst, const void* map, unsigned long long* bar, int c0, int c1, int c2) {
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
                 ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2) : "memory");
}
__device__ __forceinline__ void load4(void* dst, const void* map, unsigned long long* bar, int c0, int c1, int c2, int c3) {
    asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];"
                 ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2), "r"(c3) : "memory");
}
__device__ __forceinline__ void store3(const void* map, const void* src, int c0, int c1, int c2) {
    asm volatile("cp.async.bulk.tensor.3d.global.shared::cta.bulk_group [%0, {%2, %3, %4}], [%1];"
                 ::"l"(map), "r"(smem_u32(src)), "r"(c0), "r"(c1), "r"(c2) : "memory");
}
__device__ __forceinline__ void store4(const void* map, const void* src, int c0, int c1, int c2, int c3) {
    asm volatile("cp.async.bulk.tensor.4d.global.shared::cta.bulk_group [%0, {%2, %3, %4, %5}], [%1];"
                 ::"l"(map), "r"(smem_u32(src)), "r"(c0), "r"(c1), "r"(c2), "r"(c3) : "memory");
}
// bulk tensor store with an L2 eviction-priority hint
__device__ __forceinline__ unsigned long long make_policy_evict_last() {
    unsigned long long p;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ void store3_hint(const void* map, const void* src, int c0, int c1, int c2, unsigned long long pol) {
    asm volatile("cp.async.bulk.tensor.3d.global.shared::cta.bulk_group.L2::cache_hint [%0, {%2, %3, %4}], [%1], %5;"
                 ::"l"(map), "r"(smem_u32(src)), "r"(c0), "r"(c1), "r"(c2), "l"(pol) : "memory");
}
__device__ __forceinline__ void store_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void store_wait_read0() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void store_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
}  // namespace tma

// One 128-byte opaque CUtensorMap (kept as raw bytes so that this header needs no driver API).
struct alignas(64) TensorMapBlob { unsigned char bytes[128]; };

template <class Cfg, int TC, typename T, bool ODDFIX = false>
struct TmaTile {
    using C = cx<T>;
    static constexpr int W = (int)sizeof(C) / 8;                          // 8-byte words per element
    static constexpr int ROW_BYTES = TC * (int)sizeof(C);
    static constexpr int ROW_BYTES_WIDE = (TC + 2) * (int)sizeof(C);      // ODDFIX: landing rows of odd-l tiles
    static constexpr int PADR = (ROW_BYTES < 128 && Cfg::NST > 1 && Cfg::radix(0) % 4 == 0 &&
                                 Cfg::S % Cfg::radix(0) == 0) ? Cfg::radix(0) : 0;
    static constexpr int ROWS = Cfg::N + (PADR ? Cfg::N / PADR : 0);
    static constexpr int LAND_BYTES = Cfg::N * (ODDFIX ? ROW_BYTES_WIDE : ROW_BYTES);
    static constexpr int WORK_BYTES = ROWS * ROW_BYTES;
    static constexpr int STAGE_BYTES = (((LAND_BYTES > WORK_BYTES ? LAND_BYTES : WORK_BYTES) + 1023) / 1024) * 1024;
    static constexpr int TILE_BYTES = Cfg::N * ROW_BYTES;                 // bytes one tile moves each way
    static constexpr int TW_BYTES = ((Cfg::TWN * (int)sizeof(C) + 1023) / 1024) * 1024;
    static constexpr int NCONS = Cfg::S * TC;                             // consumer threads
    __host__ __device__ static constexpr int smem_bytes(int nstage) {
        return TW_BYTES + nstage * STAGE_BYTES + 256;
    }
    __host__ __device__ static constexpr int max_stages() {
        int n = (227 * 1024 - TW_BYTES - 256) / STAGE_BYTES;
        return n > 4 ? 4 : n;
    }
};

// The user's spectrum has rows of M+1 complex numbers.  In fp32 (8-byte elements) the rows with odd
// l = ky % (Ny/p) therefore start 8 bytes off a 16-byte boundary, and a bulk tensor copy needs 16.
// The X passes handle this (ODDFIX) by giving the tiles of odd rows a window shifted by one column on
// the user side -- columns [w*TC-1, w*TC+TC-1), which IS 16-byte aligned there -- and fetching a
// 16-byte-aligned superset (TC+2 columns) on the loading side:
//   X_FWD  load packed cols [w*TC-2, w*TC+TC) (zero-filled below 0), transform cols w*TC-1.., store the
//          aligned user window; column -1 is garbage that lands in the previous row's kz = Nz/2 slot,
//          which the Nyquist unpack kernel overwrites afterwards; the last column M-1 of an odd row is
//          covered by one extra thin tile whose single useful column is stored with plain 8-byte stores.
//   X_INV  load user cols [w*TC-1, w*TC+TC+1), transform cols w*TC.., store the aligned packed window.
// Tiles are enumerated per row pair (l even, l+1): ntz even-row tiles, then the odd-row tiles.
// X_FWD with four row classes (fp32, L % 4 == 0).  Element (l, k) of the user spectrum sits at 8-byte word
// l*(M+1) + k and M+1 = 1 (mod 4), so a 64-byte window of row l starts on a 32-byte sector iff k0 = -l (mod 4):
//   l % 4 = 0: k0 = w*TC             l % 4 = 1: k0 = w*TC - 1 (+ thin tile for column M-1)
//   l % 4 = 2: k0 = w*TC - 2, except the first window (k0 = 0, unshifted: its left neighbours are the previous
//              row's last real columns) and a thin tile for columns M-2, M-1
//   l % 4 = 3: k0 = w*TC + 1 (the last window runs into the row's own Nyquist slot) + a thin tile for column 0
// With two classes only (even / odd l) half of the windows straddle sectors; their partial sectors are read
// back from DRAM before they are written whenever the neighbouring tile is not quick enough (ncu at 2048^3:
// 50.7 GB read for 34.4).  odd = the window starts at an odd column: the loading side fetches TC+2 columns
// from k0-1.  Thin tiles store columns [c_lo, c_hi) of their window with plain stores.
struct XTile { int q, l, w, odd, thin, k0, c_lo, c_hi; };

template <int PASS, bool ODDFIX>
__device__ __forceinline__ XTile decode_xtile(long long t_id, const TmaArgs& a, int TC = 0) {
    XTile x;
    x.c_lo = 0; x.c_hi = 1;
    if constexpr (ODDFIX) {
        if (PASS == TMA_X_FWD && a.cls4) {
            const int M = a.Mp1 - 1;
            const int per_quad = 4 * a.ntz + 3;
            const long long qd = t_id / per_quad;
            int r = (int)(t_id % per_quad);
            const int quads = a.L / 4;
            x.q = (int)(qd / quads);
            const int l4 = (int)(qd % quads);
            int cls, idx;
            if (r < a.ntz) { cls = 0; idx = r; }
            else { r -= a.ntz; cls = 1 + r / (a.ntz + 1); idx = r % (a.ntz + 1); }
            x.l = 4 * l4 + cls;
            x.w = idx;
            x.thin = 0;
            if (cls == 0) x.k0 = idx * TC;
            else if (cls == 1) { x.k0 = idx * TC - 1; x.thin = idx == a.ntz; }
            else if (cls == 2) {
                if (idx == 0) x.k0 = 0;
                else if (idx < a.ntz) x.k0 = idx * TC - 2;
                else { x.k0 = M - 2; x.thin = 1; x.c_hi = 2; }
            } else {
                if (idx < a.ntz) x.k0 = idx * TC + 1;
                else { x.k0 = 1 - TC; x.thin = 1; x.c_lo = TC - 1; x.c_hi = TC; }
            }
            x.odd = x.k0 & 1;
            return x;
        }
        const int per_pair = 2 * a.ntz + (PASS == TMA_X_FWD ? 1 : 0);
        const long long pr = t_id / per_pair;
        const int r = (int)(t_id % per_pair);
        const int half = a.L / 2;
        x.odd = r >= a.ntz;
        x.w = x.odd ? r - a.ntz : r;
        x.q = (int)(pr / half);
        x.l = 2 * (int)(pr % half) + x.odd;
        x.thin = x.odd && x.w == a.ntz;
    } else {
        const long long aa = t_id / a.ntz;
        x.w = (int)(t_id % a.ntz);
        x.q = (int)(aa / a.L);
        x.l = (int)(aa % a.L);
        x.odd = 0;
        x.thin = 0;
    }
    x.k0 = x.w * TC - x.odd;
    return x;
}

template <class Cfg, int TC, int PASS, typename T, int NSTAGE, bool ODDFIX>
__global__ void __launch_bounds__(Cfg::S * TC + 32, 1)
fft_strided_tma_kernel(const __grid_constant__ TensorMapBlob in_map, const __grid_constant__ TensorMapBlob in_map2,
                       const __grid_constant__ TensorMapBlob out_map, const TmaArgs a) {
    using C = cx<T>;
    using TT = TmaTile<Cfg, TC, T, ODDFIX>;
    constexpr int P = Cfg::P, S = Cfg::S, W = TT::W, NCONS = TT::NCONS;
    constexpr int DIR = (PASS == TMA_Y_FWD || PASS == TMA_X_FWD) ? -1 : +1;
    constexpr bool XPASS = (PASS == TMA_X_FWD || PASS == TMA_X_INV);
    static_assert(!ODDFIX || XPASS, "ODDFIX is for the X passes");
    // carve: twiddles | NSTAGE stage buffers | barriers.  (No integer round-up of the base: that
    // would turn every shared-memory access into a generic-address LD/ST.)
    extern __shared__ __align__(1024) unsigned char smem_dyn[];
    C* tw = reinterpret_cast<C*>(smem_dyn);
    unsigned char* stages = smem_dyn + TT::TW_BYTES;
    unsigned long long* full = reinterpret_cast<unsigned long long*>(stages + NSTAGE * TT::STAGE_BYTES);
    unsigned long long* done = full + NSTAGE;           // consumers -> producer: tile transformed

    const int tid = threadIdx.x;
    const bool is_producer = tid >= NCONS;
    if (tid == NCONS) {
        for (int s = 0; s < NSTAGE; ++s) { tma::mbar_init(&full[s], 1); tma::mbar_init(&done[s], NCONS / 32); }
        tma::fence_mbar_init();
    }
    if (!is_producer) load_twiddles<DIR, T>(tw, reinterpret_cast<const C*>(a.tw), Cfg::TWN, tid, NCONS);
    __syncthreads();

    const long long first = blockIdx.x, stride = gridDim.x;
    const long long n_my = first < a.ntiles ? (a.ntiles - first + stride - 1) / stride : 0;

    if (is_producer) {
        if (tid != NCONS) return;
        auto issue_load = [=, &in_map, &in_map2](long long i) {
            const long long t_id = first + i * stride;
            const int s = (int)(i % NSTAGE);
            unsigned char* dst = stages + s * TT::STAGE_BYTES;
            const int nb = Cfg::N / a.in_rows;
            if constexpr (!XPASS) {
                const int tz = (int)(t_id % a.ntz);
                const int x = (int)(t_id / a.ntz);
                tma::mbar_expect_tx(&full[s], TT::TILE_BYTES);
                for (int b = 0; b < nb; ++b) {
                    void* d = dst + (size_t)b * a.in_rows * TT::ROW_BYTES;
                    const int r0 = b * a.in_rows;
                    if constexpr (PASS == TMA_Y_FWD) tma::load3(d, &in_map, &full[s], tz * TC * W, r0, x);     // natural
                    else tma::load4(d, &in_map, &full[s], tz * TC * W, r0 % a.L, x, r0 / a.L);                  // slab
                }
            } else {
                const XTile xt = decode_xtile<PASS, ODDFIX>(t_id, a, TC);
                const int rowb = xt.odd ? TT::ROW_BYTES_WIDE : TT::ROW_BYTES;
                tma::mbar_expect_tx(&full[s], (unsigned)(Cfg::N * rowb));
                for (int b = 0; b < nb; ++b) {
                    void* d = dst + (size_t)b * a.in_rows * rowb;
                    const int r0 = b * a.in_rows;
                    if constexpr (PASS == TMA_X_FWD) {           // packed slab, tile (q, l)
                        if (!xt.odd) tma::load4(d, &in_map, &full[s], xt.k0 * W, xt.l, r0, xt.q);
                        else tma::load4(d, &in_map2, &full[s], (xt.k0 - 1) * W, xt.l, r0, xt.q);
                    } else {                                     // user spectrum, rows of one (q,x) flattened
                        if (!xt.odd) tma::load3(d, &in_map, &full[s], (xt.l * a.Mp1 + xt.w * TC) * W, r0, xt.q);
                        else tma::load3(d, &in_map2, &full[s], (xt.l * a.Mp1 + xt.w * TC - 1) * W, r0, xt.q);
                    }
                }
            }
        };
        // X_FWD: half of the 64-byte windows straddle sectors of the user array; keep the partial sectors in L2
        // until the neighbouring tile completes them (otherwise they are read back from DRAM before the write)
        const unsigned long long pol_keep = tma::make_policy_evict_last();
        auto issue_store = [=, &out_map](long long i) {
            const long long t_id = first + i * stride;
            const int s = (int)(i % NSTAGE);
            const unsigned char* src = stages + s * TT::STAGE_BYTES;
            const int nb = Cfg::N / a.out_rows;
            if constexpr (!XPASS) {
                const int tz = (int)(t_id % a.ntz);
                const int x = (int)(t_id / a.ntz);
                for (int b = 0; b < nb; ++b) {
                    const void* d = src + (size_t)b * a.out_rows * TT::ROW_BYTES;
                    const int r0 = b * a.out_rows;
                    if constexpr (PASS == TMA_Y_FWD) tma::store4(&out_map, d, tz * TC * W, r0 % a.L, x, r0 / a.L);  // -> slab
                    else tma::store3(&out_map, d, tz * TC * W, r0, x);                                              // -> natural
                }
            } else {
                const XTile xt = decode_xtile<PASS, ODDFIX>(t_id, a, TC);
                if (xt.thin) return;                             // stored by the consumers
                for (int b = 0; b < nb; ++b) {
                    const void* d = src + (size_t)b * a.out_rows * TT::ROW_BYTES;
                    const int r0 = b * a.out_rows;
                    if constexpr (PASS == TMA_X_FWD)             // -> user spectrum (window shifted by -1 on odd rows)
                        tma::store3_hint(&out_map, d, (xt.l * a.Mp1 + xt.k0) * W, r0, xt.q, pol_keep);
                    else                                         // -> packed slab
                        tma::store4(&out_map, d, xt.w * TC * W, xt.l, r0, xt.q);
                }
            }
            tma::store_commit();
        };
        const long long pre = n_my < NSTAGE ? n_my : NSTAGE;
        for (long long i = 0; i < pre; ++i) issue_load(i);
        for (long long i = 0; i < n_my; ++i) {
            const int s = (int)(i % NSTAGE);
            tma::mbar_wait(&done[s], (unsigned)((i / NSTAGE) & 1));
            issue_store(i);
            if (i + NSTAGE < n_my) {
                tma::store_wait_read0();                         // slot s has been read out
                issue_load(i + NSTAGE);
            }
        }
        tma::store_wait_all();
        return;
    }

    // ---------------- consumers ----------------
    const int c = tid % TC, t = tid / TC;
    const SmLayout<TC, 0> dense{c};
    const SmLayout<TC + 2, 0> dense_wide{c + 1};                 // odd rows: TC+2 columns landed, ours is c+1
    const SmLayout<TC, TT::PADR> padded{c};
    const NamedSync<1, NCONS> sync{};
    for (long long i = 0; i < n_my; ++i) {
        const int s = (int)(i % NSTAGE);
        C* buf = reinterpret_cast<C*>(stages + s * TT::STAGE_BYTES);
        XTile xt{};
        if constexpr (XPASS) xt = decode_xtile<PASS, ODDFIX>(first + i * stride, a, TC);
        tma::mbar_wait(&full[s], (unsigned)((i / NSTAGE) & 1));
        C v[P];
        if (ODDFIX && xt.odd) read_own<Cfg, T>(v, buf, t, dense_wide);
        else read_own<Cfg, T>(v, buf, t, dense);
        if constexpr (Cfg::NST > 1) sync();                      // all inputs read: slot becomes the exchange buffer
        fft_stages<Cfg, 0, DIR, T>(v, buf, tw, t, padded, sync);
        if (PASS == TMA_X_FWD && ODDFIX && xt.thin) {
            // thin tile: only columns [c_lo, c_hi) of the window are real; plain 8-byte stores to the user's rows
            if (c >= xt.c_lo && c < xt.c_hi) {
                const long long rstride = (long long)a.L * a.Mp1;
                C* p = reinterpret_cast<C*>(a.user_out) +
                       (((long long)xt.q * a.Nx * a.L + xt.l) * a.Mp1 + (xt.k0 + c)) + t * rstride;
#pragma unroll
                for (int m = 0; m < P; ++m) { *p = v[m]; p += rstride * S; }
            }
        } else {
            if constexpr (Cfg::NST > 1) sync();                  // all exchange reads done: slot becomes the output tile
            write_own<Cfg, T>(v, buf, t, dense);
            tma::fence_proxy_async();                            // make the generic-proxy writes visible to TMA
        }
        __syncwarp();
        if ((tid & 31) == 0) tma::mbar_arrive(&done[s]);
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

template <class Cfg, int RPB, typename T, int MINB>
__global__ void __launch_bounds__(Cfg::S * RPB, MINB) fft_z_r2c_kernel(const ZArgs a) {
    using C = cx<T>;
    constexpr int P = Cfg::P, S = Cfg::S, M = Cfg::N;
    using Pad = RowPad<Cfg>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C* tw = reinterpret_cast<C*>(smem_raw);
    C* twz = tw + ((Cfg::TWN + 1) & ~1);
    C* rows = twz + M;
    load_twiddles<-1, T>(tw, reinterpret_cast<const C*>(a.tw), Cfg::TWN, threadIdx.x, blockDim.x);
    load_twiddles<-1, T>(twz, reinterpret_cast<const C*>(a.twz), M, threadIdx.x, blockDim.x);

    const int t = threadIdx.x % S, rr = threadIdx.x / S;
    const SmLayout<1, Pad::PADR> lay{rr * Pad::PITCH};
    const long long ngroups = (a.nrows + RPB - 1) / RPB;

    for (long long g = blockIdx.x; g < ngroups; g += gridDim.x) {
        const long long row = g * RPB + rr;
        const bool ok = row < a.nrows;
        // a row of Nz reals read as M (even, odd) pairs: z[m] = x[2m] + i x[2m+1]
        const C* in = reinterpret_cast<const C*>(a.in) + row * (a.in_pitch ? a.in_pitch : M);
        C* out = reinterpret_cast<C*>(a.out) + row * (a.out_pitch ? a.out_pitch : M);
        C v[P];
#pragma unroll
        for (int m = 0; m < P; ++m) v[m] = ok ? in[t + m * S] : mk<T>((T)0, (T)0);
        __syncthreads();                               // tables loaded / previous group fully read
        fft_stages<Cfg, 0, -1, T>(v, rows, tw, t, lay, CtaSync{});
        if constexpr (Cfg::NST > 1) __syncthreads();
        write_own<Cfg, T>(v, rows, t, lay);
        __syncthreads();
        // X[k] = (Z[k] + conj Z[M-k])/2 - (i/2) w^k (Z[k] - conj Z[M-k]),  w = exp(-2 pi i/Nz)
#pragma unroll
        for (int m = 0; m < P; ++m) {
            const int k = t + m * S;
            C r;
            if (k == 0) {
                r = mk<T>(v[m].x + v[m].y, v[m].x - v[m].y);          // (X[0], X[Nz/2]) packed
            } else {
                const C zm = cconj(rows[lay.at(M - k)]);
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
    load_twiddles<+1, T>(tw, reinterpret_cast<const C*>(a.tw), Cfg::TWN, threadIdx.x, blockDim.x);
    load_twiddles<+1, T>(twz, reinterpret_cast<const C*>(a.twz), M, threadIdx.x, blockDim.x);   // conj

    const int t = threadIdx.x % S, rr = threadIdx.x / S;
    const SmLayout<1, Pad::PADR> lay{rr * Pad::PITCH};
    const long long ngroups = (a.nrows + RPB - 1) / RPB;
    const T scale = (T)a.scale;

    for (long long g = blockIdx.x; g < ngroups; g += gridDim.x) {
        const long long row = g * RPB + rr;
        const bool ok = row < a.nrows;
        const C* in = reinterpret_cast<const C*>(a.in) + row * (a.in_pitch ? a.in_pitch : M);
        C* out = reinterpret_cast<C*>(a.out) + row * (a.out_pitch ? a.out_pitch : M);
        C v[P];
#pragma unroll
        for (int m = 0; m < P; ++m) v[m] = ok ? in[t + m * S] : mk<T>((T)0, (T)0);
        __syncthreads();                               // tables loaded / previous group fully read
        write_own<Cfg, T>(v, rows, t, lay);
        __syncthreads();
        // Z[k] = (X[k] + conj X[M-k]) + i conj(w)^k (X[k] - conj X[M-k]); column 0 holds the real
        // pair (X[0], X[Nz/2]): Z[0] = (X0 + XM) + i (X0 - XM).
#pragma unroll
        for (int m = 0; m < P; ++m) {
            const int k = t + m * S;
            if (k == 0) {
                v[m] = mk<T>(v[m].x + v[m].y, v[m].x - v[m].y);
            } else {
                const C xm = cconj(rows[lay.at(M - k)]);
                const C e = cadd(v[m], xm), d = csub(v[m], xm);
                const C w = cmul(twz[k], d);
                v[m] = mk<T>(e.x - w.y, e.y + w.x);
            }
        }
        if constexpr (Cfg::NST > 1) __syncthreads();
        fft_stages<Cfg, 0, +1, T>(v, rows, tw, t, lay, CtaSync{});
        // z[m] = x[2m] + i x[2m+1]; scale by 1/(Nx Ny Nz)
        if (ok) {
#pragma unroll
            for (int m = 0; m < P; ++m) out[t + m * S] = mk<T>(v[m].x * scale, v[m].y * scale);
        }
    }
}

// Plain-load C2C row kernel: rows of N complex numbers, forward or inverse (scaled) -- the z pass of 3D C2C plans
// whose rows are too short, or whose row count is not a whole number of tiles, for the bulk-pipelined kernel
// (P:81).  Same thread mapping and exchange buffer as the R2C / C2R kernels above.
template <class Cfg, int RPB, int DIR, typename T, int MINB>
__global__ void __launch_bounds__(Cfg::S * RPB, MINB) fft_z_c2c_kernel(const ZArgs a) {
    using C = cx<T>;
    constexpr int P = Cfg::P, S = Cfg::S, N = Cfg::N;
    using Pad = RowPad<Cfg>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    C* tw = reinterpret_cast<C*>(smem_raw);
    C* rows = tw + ((Cfg::TWN + 1) & ~1) + N;            // same carve as the R2C kernel (its twz table is unused here)
    load_twiddles<DIR, T>(tw, reinterpret_cast<const C*>(a.tw), Cfg::TWN, threadIdx.x, blockDim.x);

    const int t = threadIdx.x % S, rr = threadIdx.x / S;
    const SmLayout<1, Pad::PADR> lay{rr * Pad::PITCH};
    const long long ngroups = (a.nrows + RPB - 1) / RPB;
    const T scale = (T)a.scale;

    for (long long g = blockIdx.x; g < ngroups; g += gridDim.x) {
        const long long row = g * RPB + rr;
        const bool ok = row < a.nrows;
        const C* in = reinterpret_cast<const C*>(a.in) + row * (a.in_pitch ? a.in_pitch : N);
        C* out = reinterpret_cast<C*>(a.out) + row * (a.out_pitch ? a.out_pitch : N);
        C v[P];
#pragma unroll
        for (int m = 0; m < P; ++m) v[m] = ok ? in[t + m * S] : mk<T>((T)0, (T)0);
        __syncthreads();                               // tables loaded / previous group's exchange fully read
        fft_stages<Cfg, 0, DIR, T>(v, rows, tw, t, lay, CtaSync{});
        if (ok) {
#pragma unroll
            for (int m = 0; m < P; ++m) out[t + m * S] = DIR > 0 ? mk<T>(v[m].x * scale, v[m].y * scale) : v[m];
        }
    }
}

}  // namespace fft3d
