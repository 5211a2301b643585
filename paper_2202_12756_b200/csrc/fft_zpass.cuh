// fft_zpass.cuh -- passes F1 (z-axis R2C) and I3 (z-axis C2R + normalisation) on sm_100a as a
// bulk-copy pipeline:
//
//   fft_z_bulk_kernel   one persistent CTA per SM; a producer warp streams tiles of RPT contiguous
//                       rows (RPT * Nz reals = one contiguous block of global memory) through an
//                       NSTAGE-deep shared-memory ring with cp.async.bulk (1-D TMA, no tensor map);
//                       NG consumer groups of S*RPT threads each transform whole tiles IN PLACE in
//                       their ring slot and hand them back for the bulk store.
//
// Paper: step 1, z half and its reverse with the normalisation fused.
//
// A row of Nz reals is read as M = Nz/2 complex numbers z[m] = x[2m] + i x[2m+1]; S = M/P threads
// hold P points each (element k = t + m*S in v[m], on entry and on exit of the FFT).  The Hermitian
// step needs element M-k next to element k: that element lives in lane (S-t) mod S of the same row,
// register P-1-m, so it is fetched with ONE warp shuffle per word -- no shared-memory round trip.
// Only lane t = 0 pairs with itself (k = m*S <-> (P-m)*S); its P values go through a small scratch.
// exp(-2 pi i k/Nz) = exp(-2 pi i t/Nz) * exp(-2 pi i m/(2P)): one per-thread register times a
// compile-time constant instead of a table look-up per point.
#pragma once
#include <cstdint>

#include "fft_core.cuh"
#include "fft_kernels.cuh"

namespace fft3d {

struct ZBulkArgs {
    const void* in;
    void* out;
    const void* tw;              // stage twiddles of the M-point FFT (forward)
    const void* twz;             // exp(-2 pi i k / Nz), k < M
    long long ntiles;            // nrows / RPT
    double scale;                // C2R: 1/(Nx Ny Nz)
};

namespace tma {
__device__ __forceinline__ void bulk_load(void* dst, const void* src, unsigned bytes, unsigned long long* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void bulk_store(void* dst, const void* src, unsigned bytes) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;"
                 ::"l"(dst), "r"(smem_u32(src)), "r"(bytes) : "memory");
}
}  // namespace tma

// named barrier with a run-time id (one per consumer group)
struct GroupSync {
    int id, nt;
    __device__ __forceinline__ void operator()() const {
        asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nt) : "memory");
    }
};

template <class Cfg, int RPT, typename T>
struct ZTile {
    using C = cx<T>;
    static constexpr int M = Cfg::N, S = Cfg::S, P = Cfg::P;
    static constexpr int PADR = (Cfg::NST > 1) ? Cfg::radix(0) : 0;
    static constexpr int PITCH = PADR ? M + M / PADR + 1 : M;          // elements per padded row
    static constexpr int TILE_BYTES = RPT * M * (int)sizeof(C);          // bytes moved each way per tile
    static constexpr int WORK_BYTES = RPT * PITCH * (int)sizeof(C);
    static constexpr int STAGE_BYTES = ((WORK_BYTES + 1023) / 1024) * 1024;
    static constexpr int TW_BYTES = ((Cfg::TWN * (int)sizeof(C) + 1023) / 1024) * 1024;
    static constexpr int GROUP = S * RPT;                                // consumer threads per group
    static constexpr int SCRATCH_BYTES = RPT * P * (int)sizeof(C);       // lane-0 values, per group
    __host__ __device__ static constexpr int smem_bytes(int nstage, int ng) {
        return TW_BYTES + nstage * STAGE_BYTES + ng * SCRATCH_BYTES + 256;
    }
    __host__ __device__ static constexpr int max_stages(int ng) {
        int n = (227 * 1024 - TW_BYTES - ng * SCRATCH_BYTES - 256) / STAGE_BYTES;
        return n > 8 ? 8 : n;
    }
};

template <typename T>
__device__ __forceinline__ cx<T> shfl_cx(cx<T> v, int src, int width);
template <>
__device__ __forceinline__ float2 shfl_cx<float>(float2 v, int src, int width) {
    float2 r;
    r.x = __shfl_sync(0xffffffffu, v.x, src, width);
    r.y = __shfl_sync(0xffffffffu, v.y, src, width);
    return r;
}
template <>
__device__ __forceinline__ double2 shfl_cx<double>(double2 v, int src, int width) {
    double2 r;
    r.x = __shfl_sync(0xffffffffu, v.x, src, width);
    r.y = __shfl_sync(0xffffffffu, v.y, src, width);
    return r;
}

// The Hermitian step, one PAIR (k, M-k) at a time.  With e = A + conj B, d = A - conj B (A = element k, B = element
// M-k, both before the step), w = exp(-+2 pi i k/Nz) and w^(M-k) = -conj(w^k):
//   R2C (after the forward FFT):   X[k] = (e - i w d)/2,   X[M-k] = conj((e + i w d)/2)
//   C2R (before the inverse FFT):  Z[k] =  e + i w d,      Z[M-k] = conj(e - i w d)
// so the two outputs of a pair share e, d and w d: 12 operations for both instead of 12 each.  `w` arrives already
// halved for R2C.  (Scalar arithmetic on purpose, here and in the per-thread rotations of w: the operands come out of
// warp shuffles word by word; the packed f32x2 forms of fft_radix.cuh cost register moves here and were slower, measured.)
template <bool INV, typename T>
__device__ __forceinline__ void herm_pair(cx<T> a, cx<T> b, cx<T> w, cx<T>& rk, cx<T>& rmk) {
    const T ex = a.x + b.x, ey = a.y - b.y, dx = a.x - b.x, dy = a.y + b.y;
    const T wdx = w.x * dx - w.y * dy, wdy = w.x * dy + w.y * dx;
    if constexpr (!INV) {
        rk = mk<T>((T)0.5 * ex + wdy, (T)0.5 * ey - wdx);
        rmk = mk<T>((T)0.5 * ex - wdy, (T)-0.5 * ey - wdx);
    } else {
        rk = mk<T>(ex - wdy, ey + wdx);
        rmk = mk<T>(ex + wdy, wdx - ey);
    }
}

// The Hermitian step on the thread's P values, in place.  Thread t of a row holds elements k = t + m S in v[m]; element
// M-k lives in lane (S-t) mod S, register P-1-m.  Per register pair (m, m2 = P-1-m) a lane fetches the partner of its
// v[m] with one shuffle per word, computes BOTH outputs of that pair, keeps X[k] and hands X[M-k] back to the partner
// lane (whose register m2 it belongs to) with another shuffle per word -- while receiving its own v[m2] from there.
// Lane 0 pairs with itself (k = m S <-> (P-m) S, register P-m): its partners come from the scratch copy `scr` of its
// values and its second output goes to its own register P-m; its element 0 is the packed real pair (X[0], X[Nz/2]) and
// its element M/2 (register P/2) is self-conjugate.
//   INV = false: post-process after the forward FFT (wt = exp(-2 pi i t/Nz))
//   INV = true : pre-process before the inverse FFT (wt = exp(+2 pi i t/Nz))
template <class Cfg, bool INV, typename T, int MM = 0>
__device__ __forceinline__ void hermitian_rec(cx<T> (&v)[Cfg::P], cx<T> wt, int t, const cx<T>* scr) {
    using C = cx<T>;
    constexpr int P = Cfg::P, S = Cfg::S;
    if constexpr (MM < P / 2) {
        constexpr int m = MM, m2 = P - 1 - MM;
        const int src = (S - t) & (S - 1);
        const C a = v[m];
        C pa = shfl_cx<T>(v[m2], src, S);        // element M - (t + m S) = lane S-t, register P-1-m
        if constexpr (m > 0) { if (t == 0) pa = scr[P - m]; }
        // w^(t + m S) = wt * exp(-+2 pi i m/(2P))
        const C wa = mul_root<m, 2 * P, INV ? +1 : -1, T, false>(wt);
        C rk, rmk;
        herm_pair<INV, T>(a, pa, wa, rk, rmk);
        if constexpr (m == 0) { if (t == 0) rk = mk<T>(a.x + a.y, a.x - a.y); }   // (X[0], X[Nz/2]) packed / Z[0]
        const C got = shfl_cx<T>(rmk, src, S);   // X[M - (src + m S)] = my element t + m2 S, computed by lane S-t
        v[m] = rk;
        if (t != 0) v[m2] = got;
        if constexpr (m > 0) { if (t == 0) v[P - m] = rmk; }
        hermitian_rec<Cfg, INV, T, MM + 1>(v, wt, t, scr);
    }
}

template <class Cfg, bool INV, typename T>
__device__ __forceinline__ void hermitian_step(cx<T> (&v)[Cfg::P], cx<T> wt, int t, const cx<T>* scr) {
    constexpr int P = Cfg::P;
    const cx<T> mid = v[P / 2];                  // lane 0: element M/2, w^(M/2) = -+i: X = conj Z, Z = 2 conj X
    if constexpr (!INV) wt = mk<T>((T)0.5 * wt.x, (T)0.5 * wt.y);
    hermitian_rec<Cfg, INV, T>(v, wt, t, scr);
    if (t == 0) v[P / 2] = INV ? mk<T>(mid.x + mid.x, -(mid.y + mid.y)) : mk<T>(mid.x, -mid.y);
}

// DIR = -1: R2C (pass F1);  DIR = +1: C2R with normalisation (pass I3)
// C2C = true: rows of M complex numbers, plain forward / inverse (scaled) transform -- the z pass of the
// 3D C2C transform; no Hermitian step, so a row's threads need not share a warp
template <class Cfg, int RPT, int DIR, typename T, int NSTAGE, int NG, bool C2C = false>
__global__ void __launch_bounds__(Cfg::S * RPT * NG + 32, 1) fft_z_bulk_kernel(const ZBulkArgs a) {
    using C = cx<T>;
    using ZT = ZTile<Cfg, RPT, T>;
    constexpr int P = Cfg::P, S = Cfg::S, M = Cfg::N, GROUP = ZT::GROUP, NCONS = GROUP * NG;
    static_assert(C2C || (S <= 32 && (S & (S - 1)) == 0), "a row's threads must sit inside one warp");
    static_assert(GROUP % 32 == 0 && (C2C || P % 2 == 0), "group size / even P");
    extern __shared__ __align__(1024) unsigned char smem_dyn[];
    C* tw = reinterpret_cast<C*>(smem_dyn);
    unsigned char* stages = smem_dyn + ZT::TW_BYTES;
    C* scratch = reinterpret_cast<C*>(stages + NSTAGE * ZT::STAGE_BYTES);
    unsigned long long* full = reinterpret_cast<unsigned long long*>(reinterpret_cast<unsigned char*>(scratch) + NG * ZT::SCRATCH_BYTES);
    unsigned long long* done = full + NSTAGE;
    // seen[s] = number of phases of full[s] some consumer group has observed complete.  The groups use a
    // slot in turn when NSTAGE is not a multiple of NG, and a parity wait only tells the barrier's current
    // phase from the one before it: a group must not start waiting for phase n+1 before phase n is over.
    volatile int* seen = reinterpret_cast<volatile int*>(done + NSTAGE);

    const int tid = threadIdx.x;
    const bool is_producer = tid >= NCONS;
    if (tid == NCONS) {
        for (int s = 0; s < NSTAGE; ++s) { tma::mbar_init(&full[s], 1); tma::mbar_init(&done[s], GROUP / 32); seen[s] = 0; }
        tma::fence_mbar_init();
    }
    if (!is_producer) load_twiddles<DIR, T>(tw, reinterpret_cast<const C*>(a.tw), Cfg::TWN, tid, NCONS);
    __syncthreads();

    const long long first = blockIdx.x, stride = gridDim.x;
    const long long n_my = first < a.ntiles ? (a.ntiles - first + stride - 1) / stride : 0;

    if (is_producer) {
        if (tid != NCONS) return;
        const unsigned char* gin = reinterpret_cast<const unsigned char*>(a.in);
        unsigned char* gout = reinterpret_cast<unsigned char*>(a.out);
        constexpr int CHUNK = 16384;                             // bytes per bulk copy
        auto issue_load = [=](long long i) {
            const long long t_id = first + i * stride;
            const int s = (int)(i % NSTAGE);
            unsigned char* dst = stages + s * ZT::STAGE_BYTES;
            const unsigned char* src = gin + t_id * (long long)ZT::TILE_BYTES;
            tma::mbar_expect_tx(&full[s], ZT::TILE_BYTES);
            for (int o = 0; o < ZT::TILE_BYTES; o += CHUNK)
                tma::bulk_load(dst + o, src + o, ZT::TILE_BYTES - o < CHUNK ? ZT::TILE_BYTES - o : CHUNK, &full[s]);
        };
        auto issue_store = [=](long long i) {
            const long long t_id = first + i * stride;
            const int s = (int)(i % NSTAGE);
            const unsigned char* src = stages + s * ZT::STAGE_BYTES;
            unsigned char* dst = gout + t_id * (long long)ZT::TILE_BYTES;
            for (int o = 0; o < ZT::TILE_BYTES; o += CHUNK)
                tma::bulk_store(dst + o, src + o, ZT::TILE_BYTES - o < CHUNK ? ZT::TILE_BYTES - o : CHUNK);
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

    // ---------------- consumers: group g takes the CTA's tiles g, g+NG, ... ----------------
    const int g = tid / GROUP, gt = tid % GROUP;
    const int t = gt % S, rr = gt / S;                           // thread t of row rr of the tile
    const SmLayout<1, 0> dense{rr * M};
    const SmLayout<1, ZT::PADR> padded{rr * ZT::PITCH};
    const GroupSync sync{1 + g, GROUP};
    C* scr = scratch + g * (RPT * P) + rr * P;
    // exp(-2 pi i t/Nz), conjugated for the inverse
    C wt = mk<T>((T)1, (T)0);
    if constexpr (!C2C) {
        wt = reinterpret_cast<const C*>(a.twz)[t];
        if constexpr (DIR > 0) wt.y = -wt.y;
    }
    const T scale = (T)a.scale;

    for (long long i = g; i < n_my; i += NG) {
        const int s = (int)(i % NSTAGE);
        C* buf = reinterpret_cast<C*>(stages + s * ZT::STAGE_BYTES);
        const int n = (int)(i / NSTAGE);
        while (seen[s] < n) { }
        tma::mbar_wait(&full[s], (unsigned)(n & 1));
        if (gt == 0) seen[s] = n + 1;
        C v[P];
        read_own<Cfg, T>(v, buf, t, dense);
        if constexpr (DIR > 0 && !C2C) {
            if (t == 0) {
#pragma unroll
                for (int m = 0; m < P; ++m) scr[m] = v[m];
            }
            __syncwarp();
            hermitian_step<Cfg, true, T>(v, wt, t, scr);
            __syncwarp();
        }
        if constexpr (Cfg::NST > 1) sync();                      // all inputs read: slot becomes the exchange buffer
        fft_stages<Cfg, 0, DIR, T>(v, buf, tw, t, padded, sync);
        if constexpr (DIR < 0 && !C2C) {
            if (t == 0) {
#pragma unroll
                for (int m = 0; m < P; ++m) scr[m] = v[m];
            }
            __syncwarp();
            hermitian_step<Cfg, false, T>(v, wt, t, scr);
            __syncwarp();
        } else if constexpr (DIR > 0) {
#pragma unroll
            for (int m = 0; m < P; ++m) v[m] = mk<T>(v[m].x * scale, v[m].y * scale);
        }
        if constexpr (Cfg::NST > 1) sync();                      // all exchange reads done: slot becomes the output tile
        write_own<Cfg, T>(v, buf, t, dense);
        tma::fence_proxy_async();
        __syncwarp();
        if ((tid & 31) == 0) tma::mbar_arrive(&done[s]);
    }
}

}  // namespace fft3d
