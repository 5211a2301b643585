// fft_fused.cuh -- the z and y passes of one x-plane fused into ONE kernel, the plane's
// intermediate exchanged through a small L2-resident ring instead of a full HBM round trip
// (SURVEY.md 8(f)-2):
//
//   fft_zy_fused_kernel<DIR = -1>   passes F1+F2: z-axis R2C of the rows of plane x (paper step 1,
//                                   z half) -> ring -> y-axis C2C with each row ky written to
//                                   its slab address (step 1 y half + steps 2-4)
//   fft_zy_fused_kernel<DIR = +1>   passes I2+I3: the mirror image, 1/(NxNyNz) fused
//
// A 2-D FFT of a yz-plane needs a full transpose of the plane between its two 1-D stages, and a
// plane (4 MiB at 1024^2 fp32) does not fit one SM's -- or one cluster's -- shared memory.  It
// does fit the 126 MB L2 many times over.  So the kernel is a persistent dataflow pipeline over
// ALL SMs, one CTA per SM, each CTA with a fixed ROLE: "z CTAs" transform z tiles (RPT whole rows),
// "y CTAs" transform y tiles (TC columns of a plane).  Planes are handled in order; the tiles of a
// role are dealt in order to the CTAs of that role.  The "phase-1" role (forward: z, inverse: y)
// writes its result into ring slot x % R, the "phase-2" role reads it from
// there as soon as the plane is complete -- so the ring lives in L2 (written with an evict_last
// policy; the streaming input and output use evict_first) and HBM sees ONE read and ONE write of
// the array for the two passes together.
//
// Ring layout: [R][M/TC][Ny][TC] -- a plane stored column tile by column tile, so that a y tile
// (all Ny rows of TC columns) is ONE contiguous block that moves with plain bulk copies, and a z
// tile (RPT whole rows) is ONE 4-D tensor box (TC, M/TC, RPT, 1) whose shared-memory image is the
// dense [RPT][M] tile.  The transpose between the two 1-D FFTs is thus done by the TMA unit of the
// z CTAs; each role has one cheap (contiguous) and one row-granular (64-byte rows) side, instead of
// the y CTAs carrying two row-granular sides (measured: their TMA row rate was the floor).
//
// Why roles: the two tile bodies are ~35 KB of straight-line code each and the two SMs of a TPC
// share an instruction cache; with both bodies alive in one TPC 60 % of the issue stalls in the
// FFT code were instruction fetches (ncu, profiles/).  Roles follow %smid so that a TPC never mixes.  The tiles of a
// role are dealt DYNAMICALLY, in order, by an atomic counter per role (a CTA draws its next tile when a ring slot of
// its own is about to become free): no assumption about the SM ids, and a CTA that runs slower than its peers simply
// takes fewer tiles instead of holding every plane back (measured: forward 2.87 -> 2.74 ms at 1024^3).  Every spin
// on a global counter is bounded.
//
// BOTH ROLES IN EVERY CTA (FusedArgs::mixed, the default where the CTA has two consumer groups): since the packed
// arithmetic shrank the two tile bodies to ~37 KB together, a TPC's instruction cache holds both (roles mixed inside
// TPCs cost 1 % now, 50 % before), so a CTA need not be bound to one role: consumer group 0 transforms z tiles, group 1
// y tiles, and the load warp deals the ring slots to the two streams -- a phase-2 tile when its plane is complete, a
// phase-1 tile otherwise, alternating when both are possible; phase-1 tiles never hold all the slots (their stores may
// wait for the ring's back-pressure, which only phase-2 loads relieve) and are not taken a ring's depth ahead of the
// phase-2 tickets.  One exception keeps the mixed pipeline live: a CTA whose phase-2 ticket waits for plane x2 takes its
// phase-1 ticket of a plane <= x2 even into its last free slot (that very tile may be what plane x2 is waiting for, and
// the slot count is only refreshed between items).  Liveness: take the lowest phase-2 ticket not yet loaded, plane xm.
// Every phase-1 tile of xm is either in some CTA's slot -- its store waits for plane xm-R to be read out, i.e. for
// phase-2 tickets below the lowest outstanding one: all loaded -- or is the un-taken phase-1 ticket of a CTA D, and then
// xm <= D's x2, so D takes it as soon as it has a free slot; D's slots hold phase-1 tiles of planes <= xm (tickets are
// drawn in order), whose stores likewise wait only for the read-out of planes <= xm - R (all loaded), or phase-2 tiles,
// which wait for nothing.  So plane xm completes, its holder takes the ticket, and the minimum advances.
// Both groups look at every item in order and take the ones of their role.  Every SM then carries
// the same mix of compute-heavy z tiles and latency-heavy y tiles, and no SM split has to be tuned
// (measured at 1024^3: forward 2.57 -> 2.49 ms, inverse 2.82 -> 2.76 ms on the same box).
//
// Ordering between CTAs uses two counters per plane in global memory (zeroed before the launch):
//   p1_done[x]    += 1 when a phase-1 tile of plane x has been stored (store complete, released at once)
//   p2_loaded[x]  += 1 when a phase-2 tile of plane x has landed in shared memory
// A phase-2 load of plane x waits for p1_done[x] == N1; a phase-1 store of plane x waits for
// p2_loaded[x-R] == N2 (the ring slot has been read out).  Phase-2 CTAs never wait on anything a
// later plane produces and phase-1 CTAs only on phase-2 loads R planes back; tiles are drawn in plane
// order and every CTA handles its tiles in the order it drew them, so with all CTAs co-resident
// (cooperative launch) the pipeline cannot deadlock: the lowest unfinished tile of either role is
// always held by a CTA whose earlier tiles depend on lower planes only.
// End of work: a load warp that draws a tile index past the end posts NSTAGE "end items" (index -1) through the
// same barriers, so that every consumer group and every store warp sees one and leaves.
//
// Inside a CTA: a load warp, one store warp per ring slot (one elected lane each) and NG consumer groups
// that own alternate tiles and transform them IN PLACE in an NSTAGE-deep shared-memory ring, with
// exactly the z-tile and y-tile code of fft_zpass.cuh / fft_kernels.cuh.
#pragma once
#include <cstdint>

#include "fft_core.cuh"
#include "fft_kernels.cuh"
#include "fft_zpass.cuh"

namespace fft3d {

struct FusedArgs {
    const void* in;          // forward: the real input; inverse: unused (slab read through its tensor map)
    void* out;               // inverse: the real output; forward: unused (slab written through its tensor map)
    void* ring;              // [R][M/TC][Ny][TC] complex: column-tiled planes
    const void* tw_z;        // stage twiddles of the M-point FFT (forward)
    const void* twz;         // exp(-2 pi i k / Nz), k < M
    const void* tw_y;        // stage twiddles of the Ny-point FFT (forward)
    unsigned* flags;         // [2][Nx]: p1_done, p2_loaded
    int Nx, Ny, L;           // L = Ny / virtual_slabs
    int R;                   // ring planes
    int rows_slab;           // rows per TMA box on the slab side of a y tile
    double scale;            // inverse: 1/(Nx Ny Nz)
    int kz;                  // SMs [0, kz) take the z tiles (0: split by CTA pairs)
    int mixed;               // 1: every CTA runs both roles (consumer group 0 the z tiles, group 1 the y tiles)
    int jitter;              // > 0: stress option -- every load warp sleeps a pseudo-random 0..jitter ns before each item,
                             // which scrambles the order in which the CTAs draw and take their tiles (results and
                             // liveness must not depend on that order); 0 in normal use
};

namespace tma {
__device__ __forceinline__ unsigned long long policy_evict_first() {
    unsigned long long p;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ unsigned long long policy_evict_last() {
    unsigned long long p;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ void bulk_load_h(void* dst, const void* src, unsigned bytes, unsigned long long* bar,
                                            unsigned long long pol) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)), "l"(pol) : "memory");
}
__device__ __forceinline__ void bulk_store_h(void* dst, const void* src, unsigned bytes, unsigned long long pol) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group.L2::cache_hint [%0], [%1], %2, %3;"
                 ::"l"(dst), "r"(smem_u32(src)), "r"(bytes), "l"(pol) : "memory");
}
__device__ __forceinline__ void load4_h(void* dst, const void* map, unsigned long long* bar, int c0, int c1, int c2, int c3,
                                        unsigned long long pol) {
    asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%3, %4, %5, %6}], [%2], %7;"
                 ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "l"(pol) : "memory");
}
__device__ __forceinline__ void store4_h(const void* map, const void* src, int c0, int c1, int c2, int c3,
                                         unsigned long long pol) {
    asm volatile("cp.async.bulk.tensor.4d.global.shared::cta.bulk_group.L2::cache_hint [%0, {%2, %3, %4, %5}], [%1], %6;"
                 ::"l"(map), "r"(smem_u32(src)), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "l"(pol) : "memory");
}
__device__ __forceinline__ void prefetch_l2(const void* src, unsigned bytes, unsigned long long pol) {
    asm volatile("cp.async.bulk.prefetch.L2.global.L2::cache_hint [%0], %1, %2;" ::"l"(src), "r"(bytes), "l"(pol) : "memory");
}
__device__ __forceinline__ void fence_proxy_async_all() { asm volatile("fence.proxy.async;" ::: "memory"); }
}  // namespace tma
// stress option of the fused pipeline (FusedArgs::jitter): a pseudo-random pause of up to max_ns in a load warp
__device__ __forceinline__ void jitter_sleep(int max_ns, int i) {
    unsigned h = (unsigned)clock64() * 2654435761u ^ (blockIdx.x * 40503u + (unsigned)i * 977u);
    h ^= h >> 15; h *= 2246822519u; h ^= h >> 13;
    __nanosleep(h % (unsigned)max_ns);
}
namespace tma {
__device__ __forceinline__ unsigned ld_acquire(const unsigned* p) {
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void red_release_add(unsigned* p, unsigned v) {
    asm volatile("red.release.gpu.global.add.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ void red_relaxed_add(unsigned* p, unsigned v) {
    asm volatile("red.relaxed.gpu.global.add.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
// Spin on a global counter, bounded: ~1 us per poll, 2^24 polls > 10 s.  A pipeline that cannot make progress
// traps -- the host then sees a launch failure and the API returns FFT3D_ECUDA -- instead of hanging the device.
__device__ __forceinline__ void wait_count(const unsigned* p, unsigned target) {
    unsigned polls = 0;
    while (ld_acquire(p) < target) {
        __nanosleep(64);
        if (++polls > (1u << 24)) __trap();
    }
}
}  // namespace tma

template <class ZCfg, int RPT, class YCfg, int TC, typename T, int NG_ = 2>
struct FusedTile {
    using C = cx<T>;
    using ZT = ZTile<ZCfg, RPT, T>;
    using YT = TmaTile<YCfg, TC, T, false>;
    static constexpr int GROUP = ZT::GROUP;                     // consumer threads per group
    static constexpr bool OK = (ZT::GROUP == YT::NCONS) && (ZT::GROUP % 32 == 0);
    static constexpr int NG = NG_;
    static constexpr int STAGE_BYTES = ZT::STAGE_BYTES > YT::STAGE_BYTES ? ZT::STAGE_BYTES : YT::STAGE_BYTES;
    static constexpr int TWZ_BYTES = ZT::TW_BYTES, TWY_BYTES = YT::TW_BYTES;
    static constexpr int FIXED = TWZ_BYTES + TWY_BYTES + NG * ZT::SCRATCH_BYTES + 256;
    // + one load warp + one store warp per ring slot (each store thread blocks on ITS tile's completion only)
    __host__ __device__ static constexpr int threads(int nstage) { return NG * GROUP + 32 * (1 + nstage); }
    __host__ __device__ static constexpr int smem_bytes(int nstage) { return FIXED + nstage * STAGE_BYTES; }
    __host__ __device__ static constexpr int max_stages() {
        int n = (227 * 1024 - FIXED) / STAGE_BYTES;
        return n > 4 ? 4 : n;
    }
    static constexpr int THREADS = threads(max_stages());
    // Register re-allocation between the warp groups (setmaxnreg): the kernel is launched with REGS_LAUNCH registers
    // per thread (what __launch_bounds__(THREADS, 1) allows); the producer warp group (load warp + three store warps)
    // keeps REGS_PROD and the consumer warp groups take what that frees.  Only where the producers are exactly one
    // warp group and the consumers whole warp groups.
    static constexpr int NCONS_ALL = NG * GROUP;
    static constexpr int REGS_LAUNCH = ((65536 / THREADS) / 8) * 8;
    static constexpr int REGS_PROD = 32;
    static constexpr int REGS_CONS_RAW = (((REGS_LAUNCH * THREADS - 128 * REGS_PROD) / NCONS_ALL) / 8) * 8;
    static constexpr int REGS_CONS = REGS_CONS_RAW > 232 ? 232 : REGS_CONS_RAW;
    static constexpr bool REALLOC = (NCONS_ALL % 128 == 0) && (THREADS - NCONS_ALL == 128) && THREADS >= 384 &&
                                    REGS_LAUNCH <= 248 && REGS_CONS > REGS_LAUNCH;
};

// words of the control block that follows the 2*Nx plane counters in the flags area (zeroed before the launch)
enum { FZ_CTL_NZ = 0, FZ_CTL_NY = 1, FZ_CTL_ARRIVED = 2, FZ_CTL_NEXT_Z = 3, FZ_CTL_NEXT_Y = 4, FZ_CTL_WORDS = 8 };

struct FItem { int p1, x, j; };
struct TrueT { static constexpr bool value = true; };
struct FalseT { static constexpr bool value = false; };

// C2C = true: the rows are Nz complex numbers and the z tiles run the plain C2C transform (3D C2C plans)
template <class ZCfg, int RPT, class YCfg, int TC, int DIR, typename T, int NSTAGE, int NG_, bool C2C = false>
__global__ void __launch_bounds__((FusedTile<ZCfg, RPT, YCfg, TC, T, NG_>::THREADS), 1)
fft_zy_fused_kernel(const __grid_constant__ TensorMapBlob ring_map, const __grid_constant__ TensorMapBlob slab_map,
                    const FusedArgs a) {
    using C = cx<T>;
    using FT = FusedTile<ZCfg, RPT, YCfg, TC, T, NG_>;
    using ZT = typename FT::ZT;
    using YT = typename FT::YT;
    constexpr int GROUP = FT::GROUP, NG = FT::NG, NCONS = NG * GROUP, W = YT::W;
    constexpr int M = ZCfg::N, NY = YCfg::N;
    constexpr bool FWD = DIR < 0;
    static_assert(FT::OK, "z tile and y tile must use the same number of consumer threads");
    static_assert(C2C || (ZCfg::S <= 32 && (ZCfg::S & (ZCfg::S - 1)) == 0), "a row's threads must sit inside one warp");

    extern __shared__ __align__(1024) unsigned char smem_dyn[];
    C* twz_s = reinterpret_cast<C*>(smem_dyn);                                   // z stage twiddles
    C* twy_s = reinterpret_cast<C*>(smem_dyn + FT::TWZ_BYTES);                   // y stage twiddles
    unsigned char* stages = smem_dyn + FT::TWZ_BYTES + FT::TWY_BYTES;
    C* scratch = reinterpret_cast<C*>(stages + NSTAGE * FT::STAGE_BYTES);
    unsigned long long* full = reinterpret_cast<unsigned long long*>(reinterpret_cast<unsigned char*>(scratch) + NG * ZT::SCRATCH_BYTES);
    unsigned long long* done = full + NSTAGE;            // consumers -> store warp: tile transformed
    unsigned long long* empty = done + NSTAGE;           // store warp -> load warp: slot read out
    // seen[s] = number of phases of full[s] a consumer group has observed complete.  A slot is used by
    // the groups in turn (NSTAGE need not be a multiple of NG) and a parity wait is only meaningful
    // within one phase of the barrier's current one, so a group polls seen[s] before it waits for ITS phase.
    // Both roles in the CTA: every group waits on every phase, and seen[g * NSTAGE + s] counts the phases group g has
    // observed; the load warp refills slot s only when BOTH groups have observed its previous phase (a group that only
    // skips the item does not hold the slot otherwise, and a parity wait two phases late would alias).
    volatile int* seen = reinterpret_cast<volatile int*>(empty + NSTAGE);
    volatile int* role_s = seen + 2 * NSTAGE;            // [role_z] broadcast from thread 0
    volatile int* item_q = role_s + 4;                   // [s] global tile index in slot s (-1: no more tiles), [NSTAGE] first end item, [NSTAGE+1+s] its plane, [2 NSTAGE+1+s] 1 = a z tile

    const int tid = threadIdx.x;
    if (tid == NCONS) {
        for (int s = 0; s < NSTAGE; ++s) {
            tma::mbar_init(&full[s], 1); tma::mbar_init(&done[s], GROUP / 32); tma::mbar_init(&empty[s], 1);
            seen[s] = 0; seen[NSTAGE + s] = 0;
        }
        item_q[NSTAGE] = -1;
        tma::fence_mbar_init();
    }
    if (tid < NCONS) {
        load_twiddles<DIR, T>(twz_s, reinterpret_cast<const C*>(a.tw_z), ZCfg::TWN, tid, NCONS);
        load_twiddles<DIR, T>(twy_s, reinterpret_cast<const C*>(a.tw_y), YCfg::TWN, tid, NCONS);
    }
    __syncthreads();

    const int n_z = a.Ny / RPT, n_y = M / TC;            // z tiles / y tiles per plane
    const int n1 = FWD ? n_z : n_y, n2 = FWD ? n_y : n_z;
    // Role of this CTA: z tiles or y tiles, never both -- the two bodies are ~35 KB of straight-line code each,
    // and the SMs of a TPC share an instruction cache, so both SMs of a TPC get the same role: SMs [0, kz) take
    // the z tiles (kz even), the rest the y tiles; kz = 0: CTA pairs (4k, 4k+1) -> z, (4k+2, 4k+3) -> y.
    // Nothing is assumed about %smid being dense or about one CTA per SM: the tiles of a role are dealt by an
    // atomic counter (below), and the role sizes are checked after a grid-wide arrival counter (cooperative launch:
    // all CTAs are co-resident).  If a role came out empty, all CTAs fall back to alternating by blockIdx.
    unsigned* ctl = a.flags + 2 * a.Nx;
    if (tid == 0) {
        unsigned smid;
        asm("mov.u32 %0, %%smid;" : "=r"(smid));
        const int b = blockIdx.x, G = gridDim.x;
        int rz = (a.kz > 0 && a.kz < G) ? ((int)smid < a.kz) : !((b >> 1) & 1);
        atomicAdd(&ctl[rz ? FZ_CTL_NZ : FZ_CTL_NY], 1u);
        __threadfence();
        tma::red_release_add(&ctl[FZ_CTL_ARRIVED], 1u);
        tma::wait_count(&ctl[FZ_CTL_ARRIVED], (unsigned)G);
        const int nz = (int)tma::ld_acquire(&ctl[FZ_CTL_NZ]), ny = (int)tma::ld_acquire(&ctl[FZ_CTL_NY]);
        if (nz == 0 || ny == 0) rz = !(b & 1);
        role_s[0] = rz;
    }
    __syncthreads();
    const int role_z = role_s[0];
    const int my_p1 = FWD ? role_z : !role_z;            // this CTA's tiles are the phase-1 tiles
    const int nper = role_z ? n_z : n_y;                 // tiles per plane of this role
    const int total = a.Nx * nper;
    unsigned* p1_done = a.flags;
    unsigned* p2_loaded = a.flags + a.Nx;
    const long long plane_bytes = (long long)a.Ny * M * (long long)sizeof(C);

    if (tid >= NCONS) {
        if constexpr (FT::REALLOC) asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(FT::REGS_PROD));
        if (tid == NCONS) {
            // ------------------------- load warp -------------------------
            const unsigned long long pol_stream = tma::policy_evict_first(), pol_keep = tma::policy_evict_last();
            // the loads of one tile into ring slot s
            auto issue_load = [&](bool isz, int x, int j, int s) {
                unsigned char* dst = stages + s * FT::STAGE_BYTES;
                if (isz) {
                    tma::mbar_expect_tx(&full[s], ZT::TILE_BYTES);
                    if constexpr (FWD) {                 // rows of the real input (HBM stream)
                        const unsigned char* src = reinterpret_cast<const unsigned char*>(a.in) + (long long)x * plane_bytes +
                                                   (long long)j * ZT::TILE_BYTES;
                        constexpr int CHUNK = 65536;
                        for (int o = 0; o < ZT::TILE_BYTES; o += CHUNK)
                            tma::bulk_load_h(dst + o, src + o, ZT::TILE_BYTES - o < CHUNK ? ZT::TILE_BYTES - o : CHUNK, &full[s], pol_stream);
                    } else {                             // RPT rows gathered from the column-tiled ring: one box
                        tma::load4_h(dst, &ring_map, &full[s], 0, 0, j * RPT, x % a.R, pol_keep);
                    }
                } else {
                    tma::mbar_expect_tx(&full[s], YT::TILE_BYTES);
                    if constexpr (FWD) {                 // column tile j of the ring plane: one contiguous block
                        const unsigned char* src = reinterpret_cast<const unsigned char*>(a.ring) +
                                                   (long long)(x % a.R) * plane_bytes + (long long)j * YT::TILE_BYTES;
                        constexpr int CHUNK = 65536;
                        for (int o = 0; o < YT::TILE_BYTES; o += CHUNK)
                            tma::bulk_load_h(dst + o, src + o, YT::TILE_BYTES - o < CHUNK ? YT::TILE_BYTES - o : CHUNK, &full[s], pol_keep);
                    } else {                             // columns of plane x gathered from the slab layout
                        const int nb = NY / a.rows_slab;
                        for (int b = 0; b < nb; ++b) {
                            const int r0 = b * a.rows_slab;
                            tma::load4_h(dst + (size_t)b * a.rows_slab * YT::ROW_BYTES, &slab_map, &full[s],
                                         j * TC * W, r0 % a.L, x, r0 / a.L, pol_stream);
                        }
                    }
                }
            };
            if (NG == 2 && a.mixed) {
                // ---- both roles in this CTA: the load warp deals the ring slots to the two streams.  A phase-2 tile is
                // taken when its plane is complete (checked without blocking), a phase-1 tile otherwise; when both are
                // possible the streams alternate.  Phase-1 tiles never hold all the slots (their stores may wait for the
                // ring's back-pressure, which only phase-2 loads relieve) unless no phase-2 tile is left to take.
                const int tot1 = a.Nx * n1, tot2 = a.Nx * n2;
                unsigned* next1 = &ctl[FWD ? FZ_CTL_NEXT_Z : FZ_CTL_NEXT_Y];
                unsigned* next2 = &ctl[FWD ? FZ_CTL_NEXT_Y : FZ_CTL_NEXT_Z];
                int g1 = (int)atomicAdd(next1, 1u), g2 = (int)atomicAdd(next2, 1u);
                int ready = -1, inflight1 = 0, last1 = 0, ends = 0;
                unsigned p1mask = 0;                     // bit s: the item in slot s is a phase-1 tile
                for (int i = 0;; ++i) {
                    const int s = i % NSTAGE, n = i / NSTAGE;
                    if (a.jitter > 0) jitter_sleep(a.jitter, i);
                    // the readiness of the next phase-2 ticket's plane is read BEFORE the wait for the slot (an L2 round
                    // trip that would otherwise sit between the slot becoming free and its next load)
                    if (g2 < tot2) {
                        const int x2 = g2 / n2;
                        if (x2 > ready && tma::ld_acquire(&p1_done[x2]) >= (unsigned)n1) { tma::fence_proxy_async_all(); ready = x2; }
                    }
                    if (n > 0) {
                        tma::mbar_wait(&empty[s], (unsigned)((n - 1) & 1));
                        while (seen[s] < n || seen[NSTAGE + s] < n) { }      // both groups have observed the slot's last phase
                        inflight1 -= (int)((p1mask >> s) & 1u);
                        p1mask &= ~(1u << s);
                    }
                    int take = 0;                        // 1: phase-1 tile, 2: phase-2 tile, 0: nothing left
                    for (unsigned polls = 0;;) {
                        const bool has1 = g1 < tot1, has2 = g2 < tot2;
                        if (!has1 && !has2) break;
                        const int x2 = has2 ? g2 / n2 : 0x3fffffff;
                        // a phase-1 tile whose plane is a ring's depth ahead of the phase-2 tickets would only sit in
                        // its slot waiting for the ring's back-pressure: leave the slot to a phase-2 tile instead
                        const bool can1 = has1 && (!has2 || (inflight1 < NSTAGE - 1 && g1 / n1 < x2 + a.R));
                        if (can1 && (last1 == 0 || !has2)) { take = 1; break; }
                        bool can2 = has2 && x2 <= ready;
                        if (has2 && !can2 && polls > 0 && tma::ld_acquire(&p1_done[x2]) >= (unsigned)n1) {
                            tma::fence_proxy_async_all(); ready = x2; can2 = true;
                        }
                        if (can2) { take = 2; break; }
                        // LIVENESS: `inflight1` is only re-counted at the top of an iteration, so `can1` can stay false
                        // for the whole poll loop -- and the plane this CTA's phase-2 ticket waits for may be incomplete
                        // precisely because of the phase-1 ticket this CTA is holding back.  Such a ticket (plane <= x2)
                        // is taken whatever the slot count: its store waits only for phase-2 loads of plane
                        // (g1/n1 - R) < x2, i.e. for tickets below this CTA's g2, which other CTAs hold and which depend
                        // on lower planes only -- the induction of the header still closes.
                        if (can1 || (has1 && g1 / n1 <= x2)) { take = 1; break; }
                        if (polls > 0) __nanosleep(64);
                        if (++polls > (1u << 24)) __trap();
                    }
                    if (take == 0) {                     // NSTAGE end items: both groups and every store warp see one
                        item_q[s] = -1;
                        tma::mbar_arrive(&full[s]);
                        if (++ends == NSTAGE) break;
                        continue;
                    }
                    const int g = take == 1 ? g1 : g2, np = take == 1 ? n1 : n2;
                    const int x = g / np, j = g - x * np;
                    const bool isz = FWD ? take == 1 : take == 2;
                    item_q[s] = g; item_q[NSTAGE + 1 + s] = x; item_q[2 * NSTAGE + 1 + s] = isz ? 1 : 0;
                    issue_load(isz, x, j, s);
                    if (take == 1) {
                        p1mask |= 1u << s; ++inflight1; last1 = 1;
                        g1 = (int)atomicAdd(next1, 1u);
                        if constexpr (FWD) {
                            if (g1 < tot1) {
                                const int nx = g1 / n1, nj = g1 - nx * n1;
                                tma::prefetch_l2(reinterpret_cast<const unsigned char*>(a.in) + (long long)nx * plane_bytes +
                                                 (long long)nj * ZT::TILE_BYTES, ZT::TILE_BYTES, pol_stream);
                            }
                        }
                    } else {
                        last1 = 0;
                        g2 = (int)atomicAdd(next2, 1u);
                    }
                }
                return;
            }
            int i = 0, ready = -1;                       // planes <= ready are known to be complete in the ring
            unsigned* next = &ctl[role_z ? FZ_CTL_NEXT_Z : FZ_CTL_NEXT_Y];
            int g = (int)atomicAdd(next, 1u);            // the next tile of this role, in order
            for (;;) {
                const int s = i % NSTAGE, n = i / NSTAGE;
                if (a.jitter > 0) jitter_sleep(a.jitter, i);
                if (n > 0) tma::mbar_wait(&empty[s], (unsigned)((n - 1) & 1));
                if (g >= total) {                        // NSTAGE end items: every group and every store warp sees one
                    if (item_q[NSTAGE] < 0) item_q[NSTAGE] = i;
                    item_q[s] = -1;
                    tma::mbar_arrive(&full[s]);
                    if (++i >= item_q[NSTAGE] + NSTAGE) break;
                    continue;
                }
                FItem it; it.p1 = my_p1; it.x = g / nper; it.j = g - it.x * nper;
                item_q[s] = g; item_q[NSTAGE + 1 + s] = it.x; item_q[2 * NSTAGE + 1 + s] = role_z;
                if (!it.p1 && it.x > ready) {
                    tma::wait_count(&p1_done[it.x], (unsigned)n1);
                    tma::fence_proxy_async_all();
                    ready = it.x;
                }
                issue_load(FWD ? it.p1 : !it.p1, it.x, it.j, s);
                ++i;
                g = (int)atomicAdd(next, 1u);            // drawn ahead: its latency hides behind the wait for the slot
                if constexpr (FWD) {
                    // forward z tiles stream the real input from HBM with ONE load in flight per CTA (2.2-3.3 us per
                    // 64 KiB): start the next tile towards L2 now, so that its load a tile period later is an L2 hit
                    // (2.71 -> 2.50 ms at 1024^3; two tiles ahead, or the same for the inverse's slab gathers, loses)
                    if (my_p1 && g < total) {
                        const int nx = g / nper, nj = g - nx * nper;
                        tma::prefetch_l2(reinterpret_cast<const unsigned char*>(a.in) + (long long)nx * plane_bytes +
                                         (long long)nj * ZT::TILE_BYTES, ZT::TILE_BYTES, pol_stream);
                    }
                }
            }
        } else if ((tid & 31) == 0) {
            // ------------------------- store warp of ring slot my_s -------------------------
            const int my_s = (tid - NCONS) / 32 - 1;
            const unsigned long long pol_stream = tma::policy_evict_first(), pol_keep = tma::policy_evict_last();
            int freed = -1;
            for (int i = my_s;; i += NSTAGE) {
                const int s = my_s, n = i / NSTAGE;
                const unsigned char* src = stages + s * FT::STAGE_BYTES;
                tma::mbar_wait(&done[s], (unsigned)(n & 1));
                const int g = item_q[s];
                if (g < 0) break;
                const int item_z = item_q[2 * NSTAGE + 1 + s];
                FItem it; it.p1 = FWD ? item_z : !item_z; it.x = item_q[NSTAGE + 1 + s]; it.j = g - it.x * (item_z ? n_z : n_y);
                if (it.p1 && it.x >= a.R && it.x - a.R > freed) {          // ring slot must have been read out
                    tma::wait_count(&p2_loaded[it.x - a.R], (unsigned)n2);
                    freed = it.x - a.R;
                }
                const bool isz = FWD ? it.p1 : !it.p1;
                if (isz) {
                    if constexpr (FWD) {                 // RPT rows scattered into the column-tiled ring: one box
                        tma::store4_h(&ring_map, src, 0, 0, it.j * RPT, it.x % a.R, pol_keep);
                    } else {                             // rows of the real output (HBM stream)
                        unsigned char* dst = reinterpret_cast<unsigned char*>(a.out) + (long long)it.x * plane_bytes +
                                             (long long)it.j * ZT::TILE_BYTES;
                        constexpr int CHUNK = 65536;
                        for (int o = 0; o < ZT::TILE_BYTES; o += CHUNK)
                            tma::bulk_store_h(dst + o, src + o, ZT::TILE_BYTES - o < CHUNK ? ZT::TILE_BYTES - o : CHUNK, pol_stream);
                    }
                } else {
                    if constexpr (FWD) {                 // rows go to their slab addresses (steps 2-4 as addressing)
                        const int nb = NY / a.rows_slab;
                        for (int b = 0; b < nb; ++b) {
                            const int r0 = b * a.rows_slab;
                            tma::store4_h(&slab_map, src + (size_t)b * a.rows_slab * YT::ROW_BYTES,
                                          it.j * TC * W, r0 % a.L, it.x, r0 / a.L, pol_stream);
                        }
                    } else {                             // column tile j of the ring plane: one contiguous block
                        unsigned char* dst = reinterpret_cast<unsigned char*>(a.ring) +
                                             (long long)(it.x % a.R) * plane_bytes + (long long)it.j * YT::TILE_BYTES;
                        constexpr int CHUNK = 65536;
                        for (int o = 0; o < YT::TILE_BYTES; o += CHUNK)
                            tma::bulk_store_h(dst + o, src + o, YT::TILE_BYTES - o < CHUNK ? YT::TILE_BYTES - o : CHUNK, pol_keep);
                    }
                }
                tma::store_commit();
                tma::store_wait_read0();                 // slot s has been read out
                tma::mbar_arrive(&empty[s]);
                if (it.p1) {
                    // publish at once: a deferred release would make this plane's readers depend on a LATER
                    // item of this CTA, and with the ring's back-pressure that closes a cycle
                    tma::store_wait_all();
                    tma::fence_proxy_async_all();
                    tma::red_release_add(&p1_done[it.x], 1u);
                }
            }
            tma::store_wait_all();
        }
        return;
    }

    // ---------------- consumers: group gq takes the CTA's items gq, gq+NG, ... ----------------
    if constexpr (FT::REALLOC) asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(FT::REGS_CONS));
    const int gq = tid / GROUP, gt = tid % GROUP;
    const GroupSync sync{1 + gq, GROUP};
    // one loop per role (the role is fixed for the CTA's lifetime): only that role's invariants stay in registers
    auto consume = [&](auto zrole) {
        constexpr bool ISZ = decltype(zrole)::value;
        constexpr bool P1 = FWD ? ISZ : !ISZ;
        // z-tile role: thread tz of row rr;  y-tile role: thread ty of column cc
        const int tz = gt % ZCfg::S, rr = gt / ZCfg::S;
        const int cc = gt % TC, ty = gt / TC;
        const SmLayout<1, 0> z_dense{rr * M};
        const SmLayout<1, ZT::PADR> z_padded{rr * ZT::PITCH};
        const SmLayout<TC, 0> y_dense{cc};
        const SmLayout<TC, YT::PADR> y_padded{cc};
        C* scr = scratch + gq * (RPT * ZCfg::P) + rr * ZCfg::P;
        C wt = mk<T>((T)1, (T)0);                        // exp(-2 pi i t/Nz), conjugated for the inverse
        if constexpr (ISZ && !C2C) {
            wt = reinterpret_cast<const C*>(a.twz)[tz];
            if constexpr (DIR > 0) wt.y = -wt.y;
        }
        const T scale = (T)a.scale;
        const int mixed = NG == 2 ? a.mixed : 0;
        int ends = 0;
        // one role per CTA: group gq takes the CTA's items gq, gq + NG, ...; both roles in the CTA: each group looks at
        // EVERY item in order (so it observes every phase of every full[] barrier) and takes the ones of its role
        for (int i = mixed ? 0 : gq;; i += mixed ? 1 : NG) {
            const int s = i % NSTAGE, n = i / NSTAGE;
            C* buf = reinterpret_cast<C*>(stages + s * FT::STAGE_BYTES);
            if (!mixed) { while (seen[s] < n) { } }      // the previous phase of this slot has been observed
            tma::mbar_wait(&full[s], (unsigned)(n & 1));
            const int g = item_q[s];
            if (mixed && gt == 0) seen[gq * NSTAGE + s] = n + 1;
            if (mixed) {
                if (g < 0) {                             // end items: the z group hands all NSTAGE of them to the store warps
                    if (!ISZ) break;
                    __syncwarp();
                    if ((tid & 31) == 0) tma::mbar_arrive(&done[s]);
                    if (++ends == NSTAGE) break;
                    continue;
                }
                if (item_q[2 * NSTAGE + 1 + s] != (ISZ ? 1 : 0)) continue;
            } else if (g < 0) {                          // end item: pass it on to the slot's store warp
                if (gt == 0) seen[s] = n + 1;
                __syncwarp();
                if ((tid & 31) == 0) tma::mbar_arrive(&done[s]);
                if (i + NG >= item_q[NSTAGE] + NSTAGE) break;
                continue;
            }
            // (kept free of branches: a lane that leaves its warp here would stay apart for the whole tile body,
            //  and the body's warp shuffles then take the slow path for diverged warps)
            if (!mixed && gt == 0) seen[s] = n + 1;
            if constexpr (!P1) {
                // the ring tile has landed in shared memory (complete_tx observed): nothing of it can be read any
                // later, so a relaxed increment is enough to let the ring slot be overwritten
                if (gt == 0) tma::red_relaxed_add(&p2_loaded[item_q[NSTAGE + 1 + s]], 1u);
            }
            __syncwarp();
            if constexpr (ISZ) {
                constexpr int P = ZCfg::P;
                C v[P];
                read_own<ZCfg, T>(v, buf, tz, z_dense);
                if constexpr (DIR > 0 && !C2C) {
                    if (tz == 0) {
#pragma unroll
                        for (int m = 0; m < P; ++m) scr[m] = v[m];
                    }
                    __syncwarp();
                    hermitian_step<ZCfg, true, T>(v, wt, tz, scr);
                    __syncwarp();
                }
                if constexpr (ZCfg::NST > 1) sync();
                fft_stages<ZCfg, 0, DIR, T>(v, buf, twz_s, tz, z_padded, sync);
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
                    for (int m = 0; m < P; ++m) v[m] = cscale(v[m], scale);
                }
                if constexpr (ZCfg::NST > 1) sync();
                write_own<ZCfg, T>(v, buf, tz, z_dense);
            } else {
                constexpr int P = YCfg::P;
                C v[P];
                read_own<YCfg, T>(v, buf, ty, y_dense);
                if constexpr (YCfg::NST > 1) sync();
                fft_stages<YCfg, 0, DIR, T>(v, buf, twy_s, ty, y_padded, sync);
                if constexpr (YCfg::NST > 1) sync();
                write_own<YCfg, T>(v, buf, ty, y_dense);
            }
            tma::fence_proxy_async();
            __syncwarp();
            if ((tid & 31) == 0) tma::mbar_arrive(&done[s]);
        }
    };
    if ((NG == 2 && a.mixed) ? gq == 0 : role_z) consume(TrueT{}); else consume(FalseT{});
}

}  // namespace fft3d
