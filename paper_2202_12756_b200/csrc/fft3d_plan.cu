// fft3d_plan.cu -- the C ABI of include/fft3d.h: plan creation, twiddle tables, and the launch
// sequences of the forward (F1, F2, F3, fix-up) and inverse (pre-pack, I1, I2, I3) transforms.
//
// Pipeline and citations (P:n = PAPER.md line n):
//   F1  z-axis R2C on every row                        step 1, z half
//   F2  y-axis C2C, rows written to the slab layout    step 1, y half + steps 2,3,4
//   F3  x-axis C2C with stride (Ny/p)(Nz/2+1)          step 5
//   inverse: the same in reverse order with 1/(NxNyNz) fused into the last pass.
// One workspace serves both directions (optimisation 1).
#include <cuda.h>
#include <cuda_runtime.h>

#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include "../../include/fft3d.h"
#include "fft_configs.cuh"
#include "fft_kernels.cuh"
#include "fft_zpass.cuh"
#include "fft_fused.cuh"
#include "fft_split2.cuh"
#include "fft_registry.h"

namespace fft3d {

#define FFT3D_DECL(n) const KernelSet* kernelset_##n(int dtype);
FFT3D_FOREACH_N(FFT3D_DECL)
#undef FFT3D_DECL

const KernelSet* find_kernels(long long n, int dtype) {
    switch (n) {
#define FFT3D_CASE(nn) case nn: return kernelset_##nn(dtype);
        FFT3D_FOREACH_N(FFT3D_CASE)
#undef FFT3D_CASE
        default: return nullptr;
    }
}

// fix-up / pre-pack kernels (fft3d_fixup.cu)
struct PlaneArgs {
    const void* src;      // forward: unused (in place on dst); inverse: the caller's spectrum
    void* dst;            // forward: the output spectrum; inverse: side buffer [p][Nx][Ny/p]
    int Nx, Ny, L, M;     // M = Nz/2; rows of the spectrum have M+1 entries
};
cudaError_t launch_unpack_nyquist(int dtype, const PlaneArgs& a, cudaStream_t st);
struct PencilArgs {
    const void* src;
    void* dst;
    long long nrows, rows_per_a;
    int M, py, dir;
};
cudaError_t launch_pencil_convert(int dtype, const PencilArgs& a, cudaStream_t st);
cudaError_t launch_pack_nyquist(int dtype, const PlaneArgs& a, cudaStream_t st);

// the same bookkeeping for distributed plans: planes published as dense copies, own rows only (fft3d_fixup.cu)
struct DistPlaneArgs {
    const void* spec;
    void* spec_out;
    void* own;
    const void* parts[16];
    void* side;
    int Nx, Ny, L, M, q, ncols;
};
cudaError_t launch_dist_extract(int dtype, const DistPlaneArgs& a, cudaStream_t st);
cudaError_t launch_dist_unpack(int dtype, const DistPlaneArgs& a, cudaStream_t st);
cudaError_t launch_dist_pack(int dtype, const DistPlaneArgs& a, cudaStream_t st);

}  // namespace fft3d

using namespace fft3d;

struct TimingState {
    int max_calls;
    int calls[2];
    std::vector<cudaEvent_t> ev[2];      // (FFT3D_MAX_LAUNCHES + 1) events per recorded call
};

struct fft3d_plan_s {
    long long Nx, Ny, Nz, M, L;         // M = columns of the intermediate rows: Nz/2 (R2C/C2R plans), Nz (C2C plans)
    int kind;                           // 0 = R2C/C2R plan, 1 = C2C plan
    void* tw_zc;                        // stage twiddles of the C2C row kernels
    int p, dtype, esize;       // esize = bytes per real
    int variant;
    const KernelSet *kz, *ky, *kx;
    void *tw_z, *tw_y, *tw_x, *twz;     // device tables
    void* tw_zb;                        // stage twiddles of the bulk-pipelined z kernels
    int num_sms;
    int device;                // the device the plan was created on: its tables, attributes and launches belong there
    int grid_z[2], grid_y[2], grid_x[2];   // persistent grid sizes [fwd, inv]
    int grid_zp[2];                        // C2C plans: the plain-load row kernels
    bool bulk_zc;                          // C2C plans: the bulk-pipelined row kernel can run (whole tiles of long rows)
    // buffers of the host-pointer entry points (lazy)
    void *h_real, *h_cplx, *h_work;
    cudaStream_t h_stream;
    TimingState* timing;       // null unless fft3d_timing_enable was called
    // TMA-pipelined strided passes
    void* encode_fn;           // cuTensorMapEncodeTiled, resolved at run time (no libcuda link dependency)
    bool tma_y, tma_x;         // usable for this plan's extents / alignment
    bool tma_xc;               // C2C plans: TMA-pipelined x pass usable
    bool split_y;              // Y passes as two half tiles + a radix-2 combine (fft_split2.cuh)
    void* tw_y2;               // stage twiddles of the Ny/2-point transform
    bool split_x;              // X passes as two half tiles (R2C/C2R plans)
    void* tw_x2;               // stage twiddles of the Nx/2-point transform
    int x2_rows;               // rows per TMA box of the even/odd x-row views
    bool split4_x;             // X passes as four quarter tiles
    void* tw_x4;               // stage twiddles of the Nx/4-point transform
    int x4_rows;
    int y2_rows_nat, y2_rows_slab;   // rows per TMA box of the even/odd row views
    bool bulk_z;               // bulk-pipelined z kernels usable (row count a multiple of the tile)
    int y_rows_nat, y_rows_slab, x_rows;   // rows per TMA box
    // fused z+y passes (fft_fused.cuh): the workspace is [slab array | ring | side | flags]
    bool fused;                // fused kernels usable for this plan (variant 3 forces them)
    bool fused_default;        // ... and expected to win (variant 0 uses them)
    int fz_R;                  // ring depth (planes)
    int fz_kz[2];              // [fwd, inv] SMs [0, kz) run the z tiles, the others the y tiles (0: split by CTA pairs)
    int fz_mixed;              // 1: every CTA runs both roles (one consumer group each); needs two consumer groups
    int fz_R_max;              // ring planes the workspace was sized for
    int fz_jitter;             // stress option: max pause (ns) of the load warps before each item, 0 = off
    size_t slab_bytes, ring_bytes, side_bytes, flags_bytes;
    // Sub-ranges the passes work on.  A plain plan covers the whole problem; the stage entry points of a
    // distributed plan (fft3d_dist_*) run the same launch code on a copy of the plan with these narrowed.
    long long xpn;             // yz-planes handled by the z and y passes (Nx)
    long long xp0;             // index along x, in the slab array, of the first of them (0)
    long long sNx;             // x extent of one virtual-slab block of the slab array: its q stride is sNx*L*M (Nx)
    int qn;                    // virtual slabs handled by the x passes, pointers already at the first one (p)
    int dist_G, dist_rank;     // distributed plans: number of ranks and this rank (0, 0 otherwise)
    int pencil_py;             // pencil-layout plans: py (> 0), px = p; 0 otherwise
    long long nat_pitch;       // complex elements per row of the natural-layout intermediate [x][y][.]: M, or M+1 for
                               // the padded in-place layout, whose rows only the plain-load kernels can address
    int inplace;               // 1: plan of fft3d_plan_inplace (fft3d_r2c_inplace / fft3d_c2r_inplace)
};

namespace {

const long double kTwoPi = 6.283185307179586476925286766559005768L;

// exp(-2 pi i num/den), fraction reduced first
void root(long long num, long long den, long double* c, long double* s) {
    long long m = ((num % den) + den) % den;
    long double a = kTwoPi * (long double)m / (long double)den;
    *c = cosl(a);
    *s = -sinl(a);
    if (m == 0) { *c = 1; *s = 0; }
    else if (2 * m == den) { *c = -1; *s = 0; }
    else if (4 * m == den) { *c = 0; *s = -1; }
    else if (4 * m == 3 * den) { *c = 0; *s = 1; }
}

template <typename T>
void store(std::vector<unsigned char>& buf, size_t i, long double c, long double s) {
    T* p = reinterpret_cast<T*>(buf.data()) + 2 * i;
    p[0] = (T)c;
    p[1] = (T)s;
}

// Stage tables of fft_core.cuh: stage s >= 1, entry (i-1)*Ns + k = exp(-2 pi i * i*k/(Ns*r)).
int upload_stage_twiddles(int nst, const int* radix, int twn, int esize, void** dptr) {
    *dptr = nullptr;
    size_t n = (size_t)(twn > 0 ? twn : 1);
    std::vector<unsigned char> buf(n * 2 * esize, 0);
    size_t off = 0;
    long long Ns = radix[0];
    for (int s = 1; s < nst; ++s) {
        int r = radix[s];
        for (int i = 1; i < r; ++i)
            for (long long kk = 0; kk < Ns; ++kk) {
                long double c, sn;
                root((long long)i * kk, Ns * r, &c, &sn);
                if (esize == 4) store<float>(buf, off + (size_t)(i - 1) * Ns + kk, c, sn);
                else store<double>(buf, off + (size_t)(i - 1) * Ns + kk, c, sn);
            }
        off += (size_t)(r - 1) * Ns;
        Ns *= r;
    }
    if (cudaMalloc(dptr, buf.size()) != cudaSuccess) { cudaGetLastError(); return FFT3D_ENOMEM; }
    if (cudaMemcpy(*dptr, buf.data(), buf.size(), cudaMemcpyHostToDevice) != cudaSuccess) {
        cudaGetLastError();
        return FFT3D_ECUDA;
    }
    return FFT3D_OK;
}

// exp(-2 pi i k / Nz), k < M
int upload_z_twiddles(long long Nz, long long M, int esize, void** dptr) {
    *dptr = nullptr;
    std::vector<unsigned char> buf((size_t)M * 2 * esize);
    for (long long k = 0; k < M; ++k) {
        long double c, s;
        root(k, Nz, &c, &s);
        if (esize == 4) store<float>(buf, (size_t)k, c, s);
        else store<double>(buf, (size_t)k, c, s);
    }
    if (cudaMalloc(dptr, buf.size()) != cudaSuccess) { cudaGetLastError(); return FFT3D_ENOMEM; }
    if (cudaMemcpy(*dptr, buf.data(), buf.size(), cudaMemcpyHostToDevice) != cudaSuccess) {
        cudaGetLastError();
        return FFT3D_ECUDA;
    }
    return FFT3D_OK;
}

int prepare_kernel(const void* fn, int threads, size_t smem, int num_sms, int* grid) {
    if (fn == nullptr) { *grid = 0; return FFT3D_OK; }
    if (cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) {
        cudaGetLastError();
        return FFT3D_ECUDA;
    }
    int occ = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, fn, threads, smem) != cudaSuccess || occ < 1) {
        cudaGetLastError();
        return FFT3D_ECUDA;
    }
    *grid = occ * num_sms;
    return FFT3D_OK;
}

int launch(const void* fn, long long work_items, int grid_cap, int threads, size_t smem, void* args,
           cudaStream_t st) {
    if (work_items <= 0) return FFT3D_OK;
    long long g = work_items < grid_cap ? work_items : grid_cap;
    void* argv[1] = {args};
    cudaError_t e = cudaLaunchKernel(fn, dim3((unsigned)g), dim3((unsigned)threads), argv, smem, st);
    if (e != cudaSuccess) { cudaGetLastError(); return FFT3D_ECUDA; }
    return FFT3D_OK;
}

long long largest_divisor_le(long long n, long long cap) {
    for (long long d = cap < n ? cap : n; d >= 1; --d)
        if (n % d == 0) return d;
    return 1;
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// Tensor map over 8-byte words: dims[0] is the contiguous dimension, strides in bytes for dims 1..rank-1.
bool make_map(const fft3d_plan_s* pl, TensorMapBlob* out, const void* base, int rank, const long long* dims,
              const long long* strides_bytes, const int* box) {
    static_assert(sizeof(CUtensorMap) == sizeof(TensorMapBlob), "CUtensorMap is 128 bytes");
    cuuint64_t gd[5]; cuuint64_t gs[5]; cuuint32_t bx[5]; cuuint32_t es[5];
    for (int i = 0; i < rank; ++i) { gd[i] = (cuuint64_t)dims[i]; bx[i] = (cuuint32_t)box[i]; es[i] = 1; }
    for (int i = 0; i + 1 < rank; ++i) gs[i] = (cuuint64_t)strides_bytes[i];
    CUresult r = ((EncodeTiledFn)pl->encode_fn)(reinterpret_cast<CUtensorMap*>(out), CU_TENSOR_MAP_DATA_TYPE_UINT64,
                                                (cuuint32_t)rank, const_cast<void*>(base), gd, gs, bx, es,
                                                CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                                CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS;
}

// The four array views of the strided passes (sz = bytes per complex, W = sz/8 words).
bool map_natural(const fft3d_plan_s* pl, TensorMapBlob* m, const void* base, int tc, int rows) {   // [Nx][Ny][M]
    const long long sz = 2 * pl->esize, W = sz / 8;
    long long d[3] = {pl->M * W, pl->Ny, pl->xpn}, st[2] = {pl->M * sz, pl->Ny * pl->M * sz};
    int b[3] = {(int)(tc * W), rows, 1};
    return make_map(pl, m, base, 3, d, st, b);
}
bool map_slab_y(const fft3d_plan_s* pl, TensorMapBlob* m, const void* base, int tc, int rows) {    // [p][sNx][L][M], rows along (q,l)
    const long long sz = 2 * pl->esize, W = sz / 8, L = pl->L;
    // planes [xp0, xp0 + xpn) of every virtual slab: the plane coordinate of the kernels starts at 0
    const unsigned char* b0 = reinterpret_cast<const unsigned char*>(base) + (size_t)pl->xp0 * L * pl->M * sz;
    long long d[4] = {pl->M * W, L, pl->xpn, pl->p}, st[3] = {pl->M * sz, L * pl->M * sz, pl->sNx * L * pl->M * sz};
    int b[4] = {(int)(tc * W), (int)(rows < L ? rows : L), 1, (int)(rows < L ? 1 : rows / L)};
    return make_map(pl, m, b0, 4, d, st, b);
}
bool map_slab_x(const fft3d_plan_s* pl, TensorMapBlob* m, const void* base, int tc, int rows) {    // [p][Nx][L][M], rows along x; tc = box columns
    const long long sz = 2 * pl->esize, W = sz / 8, L = pl->L;
    long long d[4] = {pl->M * W, L, pl->Nx, pl->qn}, st[3] = {pl->M * sz, L * pl->M * sz, pl->Nx * L * pl->M * sz};
    int b[4] = {(int)(tc * W), 1, rows, 1};
    return make_map(pl, m, base, 4, d, st, b);
}
bool map_user_x(const fft3d_plan_s* pl, TensorMapBlob* m, const void* base, int tc, int rows, long long pitch = 0) {    // [p][Nx][L*pitch], rows along x
    const long long sz = 2 * pl->esize, W = sz / 8, L = pl->L, Mp1 = pitch > 0 ? pitch : pl->M + 1;
    long long d[3] = {L * Mp1 * W, pl->Nx, pl->qn}, st[2] = {L * Mp1 * sz, pl->Nx * L * Mp1 * sz};
    int b[3] = {(int)(tc * W), rows, 1};
    return make_map(pl, m, base, 3, d, st, b);
}

int launch_tma(const void* fn, int threads, size_t smem, int num_sms, const TensorMapBlob& in_map,
               const TensorMapBlob& in_map2, const TensorMapBlob& out_map, TmaArgs& a, cudaStream_t st) {
    long long g = a.ntiles < num_sms ? a.ntiles : num_sms;
    if (g <= 0) return FFT3D_OK;
    void* argv[4] = {(void*)&in_map, (void*)&in_map2, (void*)&out_map, (void*)&a};
    cudaError_t e = cudaLaunchKernel(fn, dim3((unsigned)g), dim3((unsigned)threads), argv, smem, st);
    if (e != cudaSuccess) { cudaGetLastError(); return FFT3D_ECUDA; }
    return FFT3D_OK;
}

int launch_zbulk(const fft3d_plan_s* pl, int d, const void* in, void* out, double scale, cudaStream_t st) {
    const KernelSet* kz = pl->kz;
    ZBulkArgs z{};
    z.in = in; z.out = out; z.tw = pl->tw_zb; z.twz = pl->twz;
    z.ntiles = pl->xpn * pl->Ny / kz->zb_rpt; z.scale = scale;
    long long g = z.ntiles < pl->num_sms ? z.ntiles : pl->num_sms;
    void* argv[1] = {&z};
    cudaError_t e = cudaLaunchKernel(kz->zb_fn[d], dim3((unsigned)g), dim3((unsigned)kz->zb_threads), argv, kz->zb_smem, st);
    if (e != cudaSuccess) { cudaGetLastError(); return FFT3D_ECUDA; }
    return FFT3D_OK;
}

// F1+F2 (d = 0: real `in` -> slab array) or I2+I3 (d = 1: slab array -> real `out`) as one cooperative launch
int launch_fused(const fft3d_plan_s* pl, int d, const void* in, void* out, void* slab, void* ring, unsigned* flags, cudaStream_t st) {
    const KernelSet* ky = pl->ky;
    const bool c2c = pl->kind == 1;
    const void* fn = c2c ? ky->fc_fn[d] : ky->fz_fn[d];
    const int f_tc = c2c ? ky->fc_tc : ky->fz_tc, f_rpt = c2c ? ky->fc_rpt : ky->fz_rpt;
    const int f_threads = c2c ? ky->fc_threads : ky->fz_threads;
    const size_t f_smem = c2c ? ky->fc_smem : ky->fz_smem;
    if (cudaMemsetAsync(flags, 0, pl->flags_bytes, st) != cudaSuccess) { cudaGetLastError(); return FFT3D_ECUDA; }
    TensorMapBlob ring_map, slab_map;
    {   // the ring as [R][M/TC][Ny][TC]; a z tile is the box (TC, M/TC, RPT, 1)
        const long long sz = 2 * pl->esize, W = sz / 8, tc = f_tc, nb = pl->M / tc;
        long long dm[4] = {tc * W, nb, pl->Ny, pl->fz_R};
        long long sb[3] = {pl->Ny * tc * sz, tc * sz, pl->Ny * pl->M * sz};
        int bx[4] = {(int)(tc * W), (int)nb, f_rpt, 1};
        if (!make_map(pl, &ring_map, ring, 4, dm, sb, bx)) return FFT3D_ECUDA;
    }
    if (!map_slab_y(pl, &slab_map, slab, f_tc, pl->y_rows_slab)) return FFT3D_ECUDA;
    FusedArgs a{};
    a.in = in; a.out = out; a.ring = ring; a.tw_z = c2c ? pl->tw_zc : pl->tw_zb; a.twz = pl->twz; a.tw_y = pl->tw_y; a.flags = flags;
    a.Nx = (int)pl->xpn; a.Ny = (int)pl->Ny; a.L = (int)pl->L; a.R = pl->fz_R; a.kz = pl->fz_kz[d];
    a.mixed = (pl->fz_mixed && (c2c ? ky->fc_ng : ky->fz_ng) == 2) ? 1 : 0;
    a.rows_slab = pl->y_rows_slab;
    a.jitter = pl->fz_jitter;
    a.scale = 1.0 / ((double)pl->Nx * (double)pl->Ny * (double)pl->Nz);
    void* argv[3] = {(void*)&ring_map, (void*)&slab_map, (void*)&a};
    cudaError_t e = cudaLaunchCooperativeKernel(fn, dim3((unsigned)pl->num_sms), dim3((unsigned)f_threads), argv, f_smem, st);
    if (e != cudaSuccess) { cudaGetLastError(); return FFT3D_ECUDA; }
    return FFT3D_OK;
}

// fp32 X_FWD: four row classes l % 4 put every user-side window on a 32-byte sector (fft_kernels.cuh, XTile)
bool x_fwd_cls4(const fft3d_plan_s* pl) {
    return pl->esize == 4 && pl->L % 4 == 0 && pl->M % 4 == 0;
}

// Y pass as two half tiles (fft_split2.cuh): d = 0 natural `in` -> slab `out`, d = 1 slab `in` -> natural `out`
int launch_y_split2(const fft3d_plan_s* pl, int d, const void* in, void* out, cudaStream_t st) {
    const KernelSet* ky = pl->ky;
    const long long sz = 2 * pl->esize, W = sz / 8, M = pl->M, L = pl->L, Ny = pl->Ny, Nx = pl->xpn;
    const int tc = ky->tma_tc;
    TensorMapBlob ev, od, mo;
    for (int h = 0; h < 2; ++h) {
        const unsigned char* base = reinterpret_cast<const unsigned char*>(in) + (size_t)h * M * sz +
                                    (d == 1 ? (size_t)pl->xp0 * L * M * sz : 0);
        bool ok;
        if (d == 0) {       // even / odd rows of [Nx][Ny][M]
            long long dm[3] = {M * W, Ny / 2, Nx}, sb[2] = {2 * M * sz, Ny * M * sz};
            int bx[3] = {(int)(tc * W), pl->y2_rows_nat, 1};
            ok = make_map(pl, h ? &od : &ev, base, 3, dm, sb, bx);
        } else {            // even / odd rows l of [p][Nx][L][M]
            const long long Lh = L / 2;
            long long dm[4] = {M * W, Lh, Nx, pl->p}, sb[3] = {2 * M * sz, L * M * sz, pl->sNx * L * M * sz};
            const int rows = pl->y2_rows_slab;
            int bx[4] = {(int)(tc * W), (int)(rows < Lh ? rows : Lh), 1, (int)(rows < Lh ? 1 : rows / Lh)};
            ok = make_map(pl, h ? &od : &ev, base, 4, dm, sb, bx);
        }
        if (!ok) return FFT3D_ECUDA;
    }
    if (!(d == 0 ? map_slab_y(pl, &mo, out, tc, pl->y_rows_slab) : map_natural(pl, &mo, out, tc, pl->y_rows_nat))) return FFT3D_ECUDA;
    TmaArgs ta{};
    ta.tw = pl->tw_y2; ta.ntz = (int)(M / tc); ta.ntiles = Nx * ta.ntz;
    ta.L = (int)L; ta.Nx = (int)pl->Nx; ta.Mp1 = (int)(M + 1);
    ta.in_rows = d == 0 ? pl->y2_rows_nat : pl->y2_rows_slab;
    ta.out_rows = d == 0 ? pl->y_rows_slab : pl->y_rows_nat;
    return launch_tma(ky->y2_fn[d], ky->y2_threads, ky->y2_smem, pl->num_sms, ev, od, mo, ta, st);
}

// X pass as two half tiles (fft_split2.cuh): d = 0 packed slab `in` -> user spectrum `out`, d = 1 the reverse
int launch_x_split2(const fft3d_plan_s* pl, int d, const void* in, void* out, cudaStream_t st) {
    const KernelSet* kx = pl->kx;
    const long long sz = 2 * pl->esize, W = sz / 8, M = pl->M, L = pl->L, Nx = pl->Nx, p = pl->qn, Mp1 = M + 1;
    const int tc = kx->tma_tc_x, rows = pl->x2_rows;
    TensorMapBlob ld[2][2], mo;          // [wide][odd x rows]
    for (int wide = 0; wide < 2; ++wide)
        for (int h = 0; h < 2; ++h) {
            const int cols = tc + 2 * wide;
            bool ok;
            if (d == 0) {       // even / odd x rows of [p][Nx][L][M]
                const unsigned char* base = reinterpret_cast<const unsigned char*>(in) + (size_t)h * L * M * sz;
                long long dm[4] = {M * W, L, Nx / 2, p}, sb[3] = {M * sz, 2 * L * M * sz, Nx * L * M * sz};
                int bx[4] = {(int)(cols * W), 1, rows, 1};
                ok = make_map(pl, &ld[wide][h], base, 4, dm, sb, bx);
            } else {            // even / odd x rows of [p][Nx][L*(M+1)]
                const unsigned char* base = reinterpret_cast<const unsigned char*>(in) + (size_t)h * L * Mp1 * sz;
                long long dm[3] = {L * Mp1 * W, Nx / 2, p}, sb[2] = {2 * L * Mp1 * sz, Nx * L * Mp1 * sz};
                int bx[3] = {(int)(cols * W), rows, 1};
                ok = make_map(pl, &ld[wide][h], base, 3, dm, sb, bx);
            }
            if (!ok) return FFT3D_ECUDA;
        }
    if (!(d == 0 ? map_user_x(pl, &mo, out, tc, pl->x_rows) : map_slab_x(pl, &mo, out, tc, pl->x_rows))) return FFT3D_ECUDA;
    TmaArgs ta{};
    ta.user_out = out;
    ta.tw = pl->tw_x2; ta.ntz = (int)(M / tc);
    ta.ntiles = (long long)p * (L / 2) * (2 * ta.ntz + (d == 0 ? 1 : 0));
    if (d == 0 && x_fwd_cls4(pl)) { ta.cls4 = 1; ta.ntiles = (long long)p * (L / 4) * (4 * ta.ntz + 3); }
    ta.L = (int)L; ta.Nx = (int)Nx; ta.Mp1 = (int)Mp1; ta.in_rows = rows; ta.out_rows = pl->x_rows;
    long long g = ta.ntiles < pl->num_sms ? ta.ntiles : pl->num_sms;
    if (g <= 0) return FFT3D_OK;
    void* argv[6] = {(void*)&ld[0][0], (void*)&ld[0][1], (void*)&ld[1][0], (void*)&ld[1][1], (void*)&mo, (void*)&ta};
    cudaError_t e = cudaLaunchKernel(kx->x2_fn[d], dim3((unsigned)g), dim3((unsigned)kx->x2_threads), argv, kx->x2_smem, st);
    if (e != cudaSuccess) { cudaGetLastError(); return FFT3D_ECUDA; }
    return FFT3D_OK;
}

// X pass as four quarter tiles (fft_split2.cuh, fft_x_split4_kernel): d = 0 packed slab -> user spectrum, d = 1 reverse
int launch_x_split4(const fft3d_plan_s* pl, int d, const void* in, void* out, cudaStream_t st) {
    const KernelSet* kx = pl->kx;
    const long long sz = 2 * pl->esize, W = sz / 8, M = pl->M, L = pl->L, Nx = pl->Nx, p = pl->qn, Mp1 = M + 1;
    const int tc = kx->tma_tc_x, rows = pl->x4_rows;
    Split4Maps maps;
    TensorMapBlob mo;
    for (int wide = 0; wide < 2; ++wide)
        for (int m = 0; m < 4; ++m) {
            const int cols = tc + 2 * wide;
            bool ok;
            if (d == 0) {
                const unsigned char* base = reinterpret_cast<const unsigned char*>(in) + (size_t)m * L * M * sz;
                long long dm[4] = {M * W, L, Nx / 4, p}, sb[3] = {M * sz, 4 * L * M * sz, Nx * L * M * sz};
                int bx[4] = {(int)(cols * W), 1, rows, 1};
                ok = make_map(pl, &maps.ld[wide][m], base, 4, dm, sb, bx);
            } else {
                const unsigned char* base = reinterpret_cast<const unsigned char*>(in) + (size_t)m * L * Mp1 * sz;
                long long dm[3] = {L * Mp1 * W, Nx / 4, p}, sb[2] = {4 * L * Mp1 * sz, Nx * L * Mp1 * sz};
                int bx[3] = {(int)(cols * W), rows, 1};
                ok = make_map(pl, &maps.ld[wide][m], base, 3, dm, sb, bx);
            }
            if (!ok) return FFT3D_ECUDA;
        }
    if (!(d == 0 ? map_user_x(pl, &mo, out, tc, pl->x_rows) : map_slab_x(pl, &mo, out, tc, pl->x_rows))) return FFT3D_ECUDA;
    TmaArgs ta{};
    ta.user_out = out;
    ta.tw = pl->tw_x4; ta.ntz = (int)(M / tc);
    ta.ntiles = (long long)p * (L / 2) * (2 * ta.ntz + (d == 0 ? 1 : 0));
    if (d == 0 && x_fwd_cls4(pl)) { ta.cls4 = 1; ta.ntiles = (long long)p * (L / 4) * (4 * ta.ntz + 3); }
    ta.L = (int)L; ta.Nx = (int)Nx; ta.Mp1 = (int)Mp1; ta.in_rows = rows; ta.out_rows = pl->x_rows;
    long long g = ta.ntiles < pl->num_sms ? ta.ntiles : pl->num_sms;
    if (g <= 0) return FFT3D_OK;
    void* argv[3] = {(void*)&maps, (void*)&mo, (void*)&ta};
    cudaError_t e = cudaLaunchKernel(kx->x4_fn[d], dim3((unsigned)g), dim3((unsigned)kx->x4_threads), argv, kx->x4_smem, st);
    if (e != cudaSuccess) { cudaGetLastError(); return FFT3D_ECUDA; }
    return FFT3D_OK;
}

// event slot `i` of the call being recorded for direction `which`, or no-op
struct Recorder {
    TimingState* t;
    int which, call;
    cudaStream_t st;
    Recorder(const fft3d_plan_s* pl, int w, cudaStream_t s) : t(pl->timing), which(w), call(-1), st(s) {
        if (t != nullptr && t->calls[w] < t->max_calls) call = t->calls[w]++;
    }
    void mark(int i) {
        if (call >= 0) cudaEventRecord(t->ev[which][(size_t)call * (FFT3D_MAX_LAUNCHES + 1) + i], st);
    }
};

bool overlap(const void* a, size_t na, const void* b, size_t nb) {
    uintptr_t x = (uintptr_t)a, y = (uintptr_t)b;
    return x < y + nb && y < x + na;
}
// a plan belongs to the device it was created on (twiddle tables, function attributes, SM count)
bool wrong_device(const fft3d_plan_s* pl) {
    int d = -1;
    if (cudaGetDevice(&d) != cudaSuccess) { cudaGetLastError(); return true; }
    return d != pl->device;
}

}  // namespace

extern "C" {

int fft3d_supported_length(long long n) {
    return find_kernels(n, FFT3D_F32) != nullptr ? 1 : 0;
}

static int plan_create(fft3d_plan_t** out, long long Nx, long long Ny, long long Nz, int dtype, int virtual_slabs, int kind) {
    if (out == nullptr) return FFT3D_EINVAL;
    *out = nullptr;
    if (dtype != FFT3D_F32 && dtype != FFT3D_F64) return FFT3D_EINVAL;
    if (Nx < 2 || Ny < 2 || Nz < 2 || virtual_slabs < 1) return FFT3D_EINVAL;
    if (Nx % virtual_slabs != 0 || Ny % virtual_slabs != 0) return FFT3D_EINVAL;
    if (kind == 0 && Nz % 2 != 0) return FFT3D_EUNSUPPORTED;
    const long long Mcols = kind == 0 ? Nz / 2 : Nz;
    const KernelSet* kz = find_kernels(Mcols, dtype);
    const KernelSet* ky = find_kernels(Ny, dtype);
    const KernelSet* kx = find_kernels(Nx, dtype);
    if (kz == nullptr || ky == nullptr || kx == nullptr) return FFT3D_EUNSUPPORTED;

    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms < 1) {
        cudaGetLastError();
        return FFT3D_ECUDA;
    }
    fft3d_plan_t* pl = new (std::nothrow) fft3d_plan_t();
    if (pl == nullptr) return FFT3D_ENOMEM;
    std::memset(pl, 0, sizeof(*pl));
    pl->Nx = Nx; pl->Ny = Ny; pl->Nz = Nz; pl->M = Mcols; pl->kind = kind; pl->p = virtual_slabs; pl->L = Ny / virtual_slabs;
    pl->dtype = dtype; pl->esize = dtype == FFT3D_F32 ? 4 : 8;
    pl->xpn = Nx; pl->xp0 = 0; pl->sNx = Nx; pl->qn = virtual_slabs; pl->nat_pitch = Mcols;
    pl->kz = kz; pl->ky = ky; pl->kx = kx; pl->num_sms = sms; pl->device = dev;

    int rc = upload_stage_twiddles(kz->nst, kz->radix, kz->twn, pl->esize, &pl->tw_z);
    if (rc == FFT3D_OK) rc = upload_stage_twiddles(ky->nst, ky->radix, ky->twn, pl->esize, &pl->tw_y);
    if (rc == FFT3D_OK) rc = upload_stage_twiddles(kx->nst, kx->radix, kx->twn, pl->esize, &pl->tw_x);
    if (rc == FFT3D_OK && kz->zb_fn[0] != nullptr)
        rc = upload_stage_twiddles(kz->zb_nst, kz->zb_radix, kz->zb_twn, pl->esize, &pl->tw_zb);
    if (rc == FFT3D_OK && kind == 0) rc = upload_z_twiddles(Nz, pl->M, pl->esize, &pl->twz);
    if (rc == FFT3D_OK && kind == 1) {
        pl->x_rows = (int)largest_divisor_le(Nx, 256);
        // rows of >= 1 KiB in whole tiles go through the bulk-pipelined row kernel, everything else (and variant 1)
        // through the plain-load one
        pl->bulk_zc = kz->zc_fn[0] != nullptr && (Nx * Ny) % kz->zc_rpt == 0;
        if (pl->bulk_zc) {
            rc = upload_stage_twiddles(kz->zc_nst, kz->zc_radix, kz->zc_twn, pl->esize, &pl->tw_zc);
            for (int d = 0; d < 2 && rc == FFT3D_OK; ++d) {
                int g = 0;
                rc = prepare_kernel(kz->zc_fn[d], kz->zc_threads, kz->zc_smem, sms, &g);
            }
        }
        for (int d = 0; d < 2 && rc == FFT3D_OK; ++d)
            rc = prepare_kernel(kz->zp_fn[d], kz->z_threads, kz->z_smem, sms, &pl->grid_zp[d]);
    }
    for (int d = 0; d < 2 && rc == FFT3D_OK; ++d) {
        rc = prepare_kernel(kz->z_fn[d], kz->z_threads, kz->z_smem, sms, &pl->grid_z[d]);
        const int ykind = d == 0 ? KIND_LIN_SLAB : KIND_SLAB_LIN;
        if (rc == FFT3D_OK) rc = prepare_kernel(ky->s_fn[d][ykind], ky->s_threads, ky->s_smem, sms, &pl->grid_y[d]);
        if (rc == FFT3D_OK) rc = prepare_kernel(kx->s_fn[d][KIND_LIN_LIN], kx->s_threads, kx->s_smem, sms, &pl->grid_x[d]);
    }
    // TMA path: needs the driver's tensor-map encoder, 16-byte strides and whole tiles
    if (rc == FFT3D_OK) {
        cudaDriverEntryPointQueryResult qres;
        void* fn = nullptr;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess ||
            qres != cudaDriverEntryPointSuccess) { cudaGetLastError(); fn = nullptr; }
        pl->encode_fn = fn;
        const long long sz = 2 * pl->esize, M = pl->M, L = pl->L;
        const bool strides_ok = (M * sz) % 16 == 0;
        pl->tma_y = pl->tma_x = false;
        if (fn != nullptr && strides_ok && ky->tma_fn[0] != nullptr && M % ky->tma_tc == 0) {
            pl->y_rows_nat = (int)largest_divisor_le(Ny, 256);
            // slab side: a box covers whole slabs (rows % L == 0) or part of one (L % rows == 0)
            long long rows = L <= 256 ? L * largest_divisor_le(pl->p, 256 / L) : largest_divisor_le(L, 256);
            pl->y_rows_slab = (int)rows;
            pl->tma_y = true;
            for (int d = 0; d < 2 && rc == FFT3D_OK; ++d) {
                int g = 0;
                rc = prepare_kernel(ky->tma_fn[d == 0 ? TMA_Y_FWD : TMA_Y_INV], ky->tma_threads, ky->tma_smem_y, sms, &g);
            }
            // whole tiles that leave room for a single ring stage: run them as two half tiles instead
            if (rc == FFT3D_OK && ky->y2_fn[0] != nullptr && L % 2 == 0) {
                const long long Lh = L / 2, H = Ny / 2;
                pl->y2_rows_nat = (int)largest_divisor_le(H, 256);
                pl->y2_rows_slab = (int)(Lh <= 256 ? Lh * largest_divisor_le(pl->p, 256 / Lh) : largest_divisor_le(Lh, 256));
                if (H % pl->y_rows_nat == 0 && H % pl->y_rows_slab == 0 && H % pl->y2_rows_slab == 0) {
                    pl->split_y = true;
                    for (int d = 0; d < 2 && rc == FFT3D_OK; ++d) {
                        int g = 0;
                        rc = prepare_kernel(ky->y2_fn[d], ky->y2_threads, ky->y2_smem, sms, &g);
                    }
                    if (rc == FFT3D_OK) rc = upload_stage_twiddles(ky->y2_nst, ky->y2_radix, ky->y2_twn, pl->esize, &pl->tw_y2);
                }
            }
        }
        if (rc == FFT3D_OK && kind == 1 && fn != nullptr && strides_ok && kx->xc_fn[0] != nullptr && M % kx->tma_tc_x == 0) {
            pl->tma_xc = true;
            for (int d = 0; d < 2 && rc == FFT3D_OK; ++d) {
                int g = 0;
                rc = prepare_kernel(kx->xc_fn[d], kx->tma_threads_x, kx->xc_smem, sms, &g);
            }
        }
        if (rc == FFT3D_OK && kind == 0 && fn != nullptr && strides_ok && kx->tma_fn[TMA_X_FWD] != nullptr && M % kx->tma_tc_x == 0 &&
            (L * (M + 1) * sz) % 16 == 0 && (!kx->tma_oddfix || L % 2 == 0)) {
            pl->x_rows = (int)largest_divisor_le(Nx, 256);
            pl->tma_x = true;
            for (int d = 0; d < 2 && rc == FFT3D_OK; ++d) {
                int g = 0;
                rc = prepare_kernel(kx->tma_fn[d == 0 ? TMA_X_FWD : TMA_X_INV], kx->tma_threads_x, kx->tma_smem_x, sms, &g);
            }
            if (rc == FFT3D_OK && kx->x4_fn[0] != nullptr && kx->tma_oddfix && Nx % 4 == 0 && (Nx / 4) % pl->x_rows == 0) {
                pl->split4_x = true;
                pl->x4_rows = (int)largest_divisor_le(Nx / 4, 256);
                for (int d = 0; d < 2 && rc == FFT3D_OK; ++d) {
                    int g = 0;
                    rc = prepare_kernel(kx->x4_fn[d], kx->x4_threads, kx->x4_smem, sms, &g);
                }
                if (rc == FFT3D_OK) rc = upload_stage_twiddles(kx->x4_nst, kx->x4_radix, kx->x4_twn, pl->esize, &pl->tw_x4);
            }
            if (rc == FFT3D_OK && kx->x2_fn[0] != nullptr && kx->tma_oddfix && Nx % 2 == 0 && (Nx / 2) % pl->x_rows == 0) {
                pl->split_x = true;
                pl->x2_rows = (int)largest_divisor_le(Nx / 2, 256);
                for (int d = 0; d < 2 && rc == FFT3D_OK; ++d) {
                    int g = 0;
                    rc = prepare_kernel(kx->x2_fn[d], kx->x2_threads, kx->x2_smem, sms, &g);
                }
                if (rc == FFT3D_OK) rc = upload_stage_twiddles(kx->y2_nst, kx->y2_radix, kx->y2_twn, pl->esize, &pl->tw_x2);
            }
        }
    }
    if (rc == FFT3D_OK && kind == 0 && kz->zb_fn[0] != nullptr && (Nx * Ny) % kz->zb_rpt == 0) {
        pl->bulk_z = true;
        for (int d = 0; d < 2 && rc == FFT3D_OK; ++d) {
            int g = 0;
            rc = prepare_kernel(kz->zb_fn[d], kz->zb_threads, kz->zb_smem, sms, &g);
        }
    }
    // fused z+y passes: cubic-like extents, whole tiles, a ring of >= 3 planes inside ~48 MB of L2,
    // and a device that can hold one CTA per SM co-resident (cooperative launch)
    pl->slab_bytes = (size_t)Nx * Ny * pl->M * 2 * pl->esize;
    if (rc == FFT3D_OK && kind == 0 && pl->tma_y && pl->bulk_z && ky->fz_fn[0] != nullptr && Nz == Ny && ky->fz_tc == ky->tma_tc &&
        Ny % ky->fz_rpt == 0 && pl->M % ky->fz_tc == 0 && pl->M / ky->fz_tc <= 256) {
        const size_t plane = (size_t)Ny * pl->M * 2 * pl->esize;
        int R = (int)(((size_t)48 << 20) / plane);
        if (R > 8) R = 8;
        int coop = 0;
        cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev);
        if (R >= 2 && Nx >= R && coop) {
            bool ok = true;
            for (int d = 0; d < 2 && ok; ++d) {
                int g = 0;
                ok = prepare_kernel(ky->fz_fn[d], ky->fz_threads, ky->fz_smem, sms, &g) == FFT3D_OK && g >= sms;
            }

            if (ok) {
                pl->fused = true; pl->fz_R = pl->fz_R_max = R; pl->fz_mixed = 1;
                // a z tile costs more than a y tile (Hermitian step, HBM-side latency): 57 % of the SMs (84 of 148: best
                // of a sweep 72..96 in both directions with the round-2 kernels; 80 before), rounded to whole TPCs
                pl->fz_kz[0] = pl->fz_kz[1] = (int)(sms * 0.57 + 0.5) & ~1;
                // measured on B200: the fused pass wins once the array is far larger than L2 and the CTA has
                // two consumer groups on a 3-slot ring (fp32 1024^3: 2.64 vs 3.13 ms); below that the
                // counters' latency and the single group (fp64: 2 slots) cost more than the HBM pass saved
                pl->fused_default = ky->fz_ng >= 2 && ky->fz_nstage >= 3 && pl->slab_bytes >= ((size_t)2 << 30);
                pl->ring_bytes = plane * R;
                pl->side_bytes = ((size_t)Nx * Ny * 2 * pl->esize + 255) & ~(size_t)255;
                pl->flags_bytes = (((size_t)2 * Nx + FZ_CTL_WORDS) * sizeof(unsigned) + 255) & ~(size_t)255;
            }
        }
    }
    // C2C plans: the same fused pipeline over rows of Nz complex points (Nz == Ny)
    if (rc == FFT3D_OK && kind == 1 && pl->tma_y && ky->fc_fn[0] != nullptr && Nz == Ny && ky->fc_tc == ky->tma_tc &&
        Ny % ky->fc_rpt == 0 && pl->M % ky->fc_tc == 0 && pl->M / ky->fc_tc <= 256 && pl->bulk_zc) {
        const size_t plane = (size_t)Ny * pl->M * 2 * pl->esize;
        int R = (int)(((size_t)48 << 20) / plane);
        if (R > 8) R = 8;
        int coop = 0;
        cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev);
        if (R >= 2 && Nx >= R && coop) {
            bool ok = true;
            for (int d = 0; d < 2 && ok; ++d) {
                int g = 0;
                ok = prepare_kernel(ky->fc_fn[d], ky->fc_threads, ky->fc_smem, sms, &g) == FFT3D_OK && g >= sms;
            }

            if (ok) {
                pl->fused = true; pl->fz_R = pl->fz_R_max = R; pl->fz_mixed = 1;
                pl->fz_kz[0] = pl->fz_kz[1] = (sms / 2 + 1) & ~1;      // z and y tiles cost about the same here
                pl->fused_default = pl->slab_bytes >= ((size_t)2 << 30);
                pl->ring_bytes = plane * R;
                pl->flags_bytes = (((size_t)2 * Nx + FZ_CTL_WORDS) * sizeof(unsigned) + 255) & ~(size_t)255;
            }
        }
    }
    if (rc != FFT3D_OK) { fft3d_destroy(pl); return rc; }
    *out = pl;
    return FFT3D_OK;
}

int fft3d_plan(fft3d_plan_t** out, long long Nx, long long Ny, long long Nz, int dtype, int virtual_slabs) {
    return plan_create(out, Nx, Ny, Nz, dtype, virtual_slabs, 0);
}
// Pencil layout: px x py virtual ranks.  The transform is the slab transform with p = px; its rows
// are then cut into the py column ranges (one more pass over the spectrum, fft3d_fixup.cu).
int fft3d_plan_pencil(fft3d_plan_t** out, long long Nx, long long Ny, long long Nz, int dtype, int px, int py) {
    if (out == nullptr) return FFT3D_EINVAL;
    *out = nullptr;
    if (px < 1 || py < 1 || py > 64) return FFT3D_EINVAL;
    // (Nx/px) x (Ny/py) x Nz pencils in real space, kz = 0..Nz/2-1 in py equal ranges (+ the Nyquist column)
    if (Nz >= 2 && Nz % 2 == 0 && (Ny % py != 0 || (Nz / 2) % py != 0)) return FFT3D_EINVAL;
    int rc = plan_create(out, Nx, Ny, Nz, dtype, px, 0);                // checks px | Nx and px | Ny
    if (rc != FFT3D_OK) return rc;
    (*out)->pencil_py = py;
    return FFT3D_OK;
}
int fft3d_plan_c2c(fft3d_plan_t** out, long long Nx, long long Ny, long long Nz, int dtype, int virtual_slabs) {
    return plan_create(out, Nx, Ny, Nz, dtype, virtual_slabs, 1);
}

size_t fft3d_workspace_bytes(const fft3d_plan_t* pl) {
    if (pl == nullptr) return 0;
    const size_t base = pl->slab_bytes + pl->ring_bytes + pl->side_bytes + pl->flags_bytes;
    // pencil-layout plans stage the slab-layout spectrum behind the ordinary workspace
    return pl->pencil_py > 0 ? ((base + 255) & ~(size_t)255) + fft3d_complex_bytes(pl) : base;
}
size_t fft3d_real_bytes(const fft3d_plan_t* pl) {
    return (pl && pl->kind == 0) ? (size_t)pl->Nx * pl->Ny * pl->Nz * pl->esize : 0;
}
size_t fft3d_complex_bytes(const fft3d_plan_t* pl) {
    if (pl == nullptr) return 0;
    return (size_t)pl->Nx * pl->Ny * (pl->kind == 0 ? pl->M + 1 : pl->Nz) * 2 * pl->esize;
}

long long fft3d_index(const fft3d_plan_t* pl, long long kx, long long ky, long long kz) {
    if (pl == nullptr || kx < 0 || kx >= pl->Nx || ky < 0 || ky >= pl->Ny || kz < 0) return -1;
    const long long pitch = pl->kind == 0 ? pl->M + 1 : pl->Nz;
    if (kz >= pitch) return -1;
    const long long q = ky / pl->L, l = ky % pl->L;
    if (pl->pencil_py > 0) {                               // blocks [a = q][b]; block (a, b) is [Nx][Ny/px][cz_b]
        const long long c = pl->M / pl->pencil_py;
        long long b = kz / c;
        if (b > pl->pencil_py - 1) b = pl->pencil_py - 1;
        const long long cz = b == pl->pencil_py - 1 ? c + 1 : c;
        return q * pl->Nx * pl->L * pitch + b * pl->Nx * pl->L * c + (kx * pl->L + l) * cz + (kz - b * c);
    }
    return ((q * pl->Nx + kx) * pl->L + l) * pitch + kz;
}

static bool use_fused(const fft3d_plan_t* pl) {
    if (pl->nat_pitch != pl->M) return false;
    return (pl->variant == 0 && pl->fused_default) || (pl->variant == 3 && pl->fused);
}
static bool use_tma(const fft3d_plan_t* pl) { return pl->variant != 1; }

// Which implementation each pass of an R2C/C2R plan runs with the current variant (one place: the launch
// code below and fft3d_launch_impl both ask these).
enum PassImpl { IMPL_PLAIN = 0, IMPL_TMA, IMPL_TMA_SPLIT2, IMPL_TMA_SPLIT4, IMPL_BULK, IMPL_FUSED, IMPL_FIXUP };
static PassImpl z_impl(const fft3d_plan_t* pl) { return use_tma(pl) && pl->bulk_z && pl->nat_pitch == pl->M ? IMPL_BULK : IMPL_PLAIN; }
static PassImpl y_impl(const fft3d_plan_t* pl) {
    if (pl->nat_pitch != pl->M) return IMPL_PLAIN;         // rows of M+1 fp32 complex are not 16-byte aligned: no TMA
    if (use_tma(pl) && pl->split_y && pl->variant != 2) return IMPL_TMA_SPLIT2;
    return use_tma(pl) && pl->tma_y ? IMPL_TMA : IMPL_PLAIN;
}
static PassImpl x_impl(const fft3d_plan_t* pl, int d) {
    if (pl->kind == 1) return use_tma(pl) && pl->tma_xc ? IMPL_TMA : IMPL_PLAIN;
    if (!(use_tma(pl) && pl->tma_x)) return IMPL_PLAIN;
    // (the quarter-tile kernel is used for the inverse only: measured at 2048^3, F3 25.1 ms against 23.4 ms whole
    // tiles -- its thin tiles cost four loads each -- but I1 20.0 against 22.8)
    if (d == 1 && pl->split4_x && pl->variant != 2) return IMPL_TMA_SPLIT4;
    if (pl->split_x && pl->variant != 2) return IMPL_TMA_SPLIT2;
    return IMPL_TMA;
}

int fft3d_launches(const fft3d_plan_t* pl, int which) {
    if (pl == nullptr || which < 0 || which > 1) return 0;
    if (pl->kind == 1) return use_fused(pl) ? 2 : 3;
    // c2r on the TMA path runs the packed column 0 of the x pass as a separate small kernel
    int n = (which == 1 && use_tma(pl) && pl->tma_x) ? 5 : 4;
    if (pl->pencil_py > 0) ++n;                  // pencil_split (last) / pencil_merge (first)
    return use_fused(pl) ? n - 1 : n;
}

const char* fft3d_launch_name(const fft3d_plan_t* pl, int which, int i) {
    if (pl == nullptr || i < 0 || i >= fft3d_launches(pl, which)) return nullptr;
    if (pl->kind == 1) {
        static const char* const cf[] = {"z_c2c_fwd", "y_c2c_fwd", "x_c2c_fwd"};
        static const char* const ci[] = {"x_c2c_inv", "y_c2c_inv", "z_c2c_inv"};
        static const char* const ff[] = {"zy_c2c_fused_fwd", "x_c2c_fwd"};
        static const char* const fi[] = {"x_c2c_inv", "yz_c2c_fused_inv"};
        if (use_fused(pl)) return which == 0 ? ff[i] : fi[i];
        return which == 0 ? cf[i] : ci[i];
    }
    const bool fz = use_fused(pl);
    if (which == 0) {
        static const char* const u[] = {"z_r2c", "y_c2c_fwd", "x_c2c_fwd", "nyquist_unpack", "pencil_split"};
        static const char* const f[] = {"zy_r2c_fused", "x_c2c_fwd", "nyquist_unpack", "pencil_split"};
        return fz ? f[i] : u[i];
    }
    const bool col0 = use_tma(pl) && pl->tma_x;
    const char* seq[6];
    int n = 0;
    if (pl->pencil_py > 0) seq[n++] = "pencil_merge";
    seq[n++] = "nyquist_pack";
    seq[n++] = "x_c2c_inv";
    if (col0) seq[n++] = "x_c2c_inv_col0";
    if (fz) seq[n++] = "yz_c2r_fused";
    else { seq[n++] = "y_c2c_inv"; seq[n++] = "z_c2r"; }
    return seq[i];
}

const char* fft3d_launch_impl(const fft3d_plan_t* pl, int which, int i) {
    const char* nm = fft3d_launch_name(pl, which, i);
    if (nm == nullptr) return nullptr;
    static const char* const names[] = {"plain", "tma", "tma_split2", "tma_split4", "bulk", "fused_ring", "fixup"};
    PassImpl im = IMPL_FIXUP;
    if (std::strstr(nm, "fused") != nullptr) im = IMPL_FUSED;
    else if (std::strncmp(nm, "pencil", 6) == 0) im = IMPL_FIXUP;
    else if (std::strcmp(nm, "x_c2c_inv_col0") == 0) im = IMPL_PLAIN;
    else if (nm[0] == 'z') im = pl->kind == 1 ? (use_tma(pl) && pl->bulk_zc ? IMPL_BULK : IMPL_PLAIN) : z_impl(pl);
    else if (nm[0] == 'y') im = y_impl(pl);
    else if (nm[0] == 'x') im = x_impl(pl, which);
    return names[im];
}

int fft3d_set_option(fft3d_plan_t* pl, int option, long long value) {
    if (pl == nullptr) return FFT3D_EINVAL;
    switch (option) {
        case FFT3D_OPT_FUSED_Z_SMS_FWD:
        case FFT3D_OPT_FUSED_Z_SMS_INV:
            if (value < 0 || value >= pl->num_sms || (value & 1)) return FFT3D_EINVAL;   // whole TPCs; 0 = split by CTA pairs
            pl->fz_kz[option == FFT3D_OPT_FUSED_Z_SMS_FWD ? 0 : 1] = (int)value;
            return FFT3D_OK;
        case FFT3D_OPT_FUSED_MIXED:
            if (value != 0 && value != 1) return FFT3D_EINVAL;
            pl->fz_mixed = (int)value;
            return FFT3D_OK;
        case FFT3D_OPT_FUSED_JITTER:
            if (value < 0 || value > 1000000) return FFT3D_EINVAL;
            pl->fz_jitter = (int)value;
            return FFT3D_OK;
        case FFT3D_OPT_FUSED_RING_PLANES:
            if (!pl->fused || value < 2 || value > pl->fz_R_max || value > pl->Nx) return FFT3D_EINVAL;
            pl->fz_R = (int)value;
            return FFT3D_OK;
        default:
            return FFT3D_EINVAL;
    }
}

int fft3d_set_variant(fft3d_plan_t* pl, int variant) {
    // 0 = the fastest known path (fused z+y passes where they win, TMA-pipelined passes elsewhere),
    // 1 = plain-load kernels only, 2 = unfused TMA-pipelined passes (six array passes per pair),
    // 3 = fused z+y passes wherever they are compiled
    if (pl == nullptr || variant < 0 || variant > 3) return FFT3D_EINVAL;
    pl->variant = variant;
    return FFT3D_OK;
}

// ---- the stages of the R2C / C2R pipelines, on the plan's sub-ranges (whole problem for a plain plan) ----

// F1 + F2 (paper step 1 and steps 2-4) of planes [xp0, xp0 + xpn): real `d_in` -> slab array.
// Fused: through `ring` (L2) with the plane counters in `flags`; unfused: through `scratch` [xpn][Ny][M].
static int stage_fwd_zy(const fft3d_plan_t* pl, const void* d_in, void* scratch, void* slab, void* ring, unsigned* flags,
                        cudaStream_t st, Recorder& rec, int& slot) {
    const long long Nxp = pl->xpn, Ny = pl->Ny, M = pl->M, L = pl->L;
    int rc;
    if (use_fused(pl)) {
        rc = launch_fused(pl, 0, d_in, nullptr, slab, ring, flags, st);
        rec.mark(slot++);
        return rc;
    }
    // F1: real [xpn*Ny rows][Nz] -> packed complex [xpn][Ny][M] in the scratch
    const KernelSet* kz = pl->kz;
    ZArgs z{};
    z.in = d_in; z.out = scratch; z.tw = pl->tw_z; z.twz = pl->twz; z.nrows = Nxp * Ny; z.scale = 1.0;
    z.in_pitch = z.out_pitch = pl->nat_pitch;
    if (z_impl(pl) == IMPL_BULK) rc = launch_zbulk(pl, 0, d_in, scratch, 1.0, st);
    else rc = launch(kz->z_fn[0], (z.nrows + kz->z_rpb - 1) / kz->z_rpb, pl->grid_z[0], kz->z_threads, kz->z_smem, &z, st);
    if (rc != FFT3D_OK) return rc;
    rec.mark(slot++);

    // F2: y-axis FFT of the scratch [x][y][M]; row ky goes to slab[q][xp0 + x][ky_l][M]  (steps 2-4 folded in)
    const KernelSet* ky = pl->ky;
    if (y_impl(pl) == IMPL_TMA_SPLIT2) {
        rc = launch_y_split2(pl, 0, scratch, slab, st);
    } else if (y_impl(pl) == IMPL_TMA) {
        TensorMapBlob mi, mo;
        if (!map_natural(pl, &mi, scratch, ky->tma_tc, pl->y_rows_nat) ||
            !map_slab_y(pl, &mo, slab, ky->tma_tc, pl->y_rows_slab)) return FFT3D_ECUDA;
        TmaArgs ta{};
        ta.tw = pl->tw_y; ta.ntz = (int)(M / ky->tma_tc); ta.ntiles = Nxp * ta.ntz;
        ta.L = (int)L; ta.Nx = (int)pl->Nx; ta.Mp1 = (int)(M + 1); ta.in_rows = pl->y_rows_nat; ta.out_rows = pl->y_rows_slab;
        rc = launch_tma(ky->tma_fn[TMA_Y_FWD], ky->tma_threads, ky->tma_smem_y, pl->num_sms, mi, mi, mo, ta, st);
    } else {
        StridedArgs a{};
        a.in = scratch; a.col0 = nullptr; a.tw = pl->tw_y;
        a.out = reinterpret_cast<unsigned char*>(slab) + (size_t)pl->xp0 * L * M * 2 * pl->esize;
        a.ntz = (int)((M + ky->tc - 1) / ky->tc); a.ncols = (int)M; a.a_lo = 1; a.L = (int)L;
        a.ntiles = Nxp * a.ntz;
        a.in_hi = Ny * pl->nat_pitch; a.in_lo = 0; a.in_rq = 0; a.in_rl = pl->nat_pitch;
        a.out_hi = L * M; a.out_lo = 0; a.out_rq = pl->sNx * L * M; a.out_rl = M;
        rc = launch(ky->s_fn[0][KIND_LIN_SLAB], a.ntiles, pl->grid_y[0], ky->s_threads, ky->s_smem, &a, st);
    }
    rec.mark(slot++);
    return rc;
}

// F3 (paper step 5): x-axis FFT inside each of the qn virtual slabs: slab (pitch M) -> spectrum (pitch M+1).
static int stage_fwd_x(const fft3d_plan_t* pl, const void* slab, void* d_out, cudaStream_t st, Recorder& rec, int& slot) {
    const long long Nx = pl->Nx, M = pl->M, L = pl->L, p = pl->qn;
    const KernelSet* kx = pl->kx;
    int rc;
    if (x_impl(pl, 0) == IMPL_TMA_SPLIT2) {
        rc = launch_x_split2(pl, 0, slab, d_out, st);
    } else if (x_impl(pl, 0) == IMPL_TMA) {
        TensorMapBlob mi, mo;
        TensorMapBlob mi2;
        const int tc = kx->tma_tc_x, of = kx->tma_oddfix;
        if (!map_slab_x(pl, &mi, slab, tc, pl->x_rows) || !map_slab_x(pl, &mi2, slab, tc + 2, pl->x_rows) ||
            !map_user_x(pl, &mo, d_out, tc, pl->x_rows)) return FFT3D_ECUDA;
        TmaArgs ta{};
        ta.user_out = d_out;
        ta.tw = pl->tw_x; ta.ntz = (int)(M / tc);
        ta.ntiles = of ? (long long)p * (L / 2) * (2 * ta.ntz + 1) : (long long)p * L * ta.ntz;
        if (of && x_fwd_cls4(pl)) { ta.cls4 = 1; ta.ntiles = (long long)p * (L / 4) * (4 * ta.ntz + 3); }
        ta.L = (int)L; ta.Nx = (int)Nx; ta.Mp1 = (int)(M + 1); ta.in_rows = pl->x_rows; ta.out_rows = pl->x_rows;
        rc = launch_tma(kx->tma_fn[TMA_X_FWD], kx->tma_threads_x, kx->tma_smem_x, pl->num_sms, mi, mi2, mo, ta, st);
    } else {
        StridedArgs b{};
        b.in = slab; b.out = d_out; b.col0 = nullptr; b.tw = pl->tw_x;
        b.ntz = (int)((M + kx->tc - 1) / kx->tc); b.ncols = (int)M; b.a_lo = (int)L; b.L = (int)Nx;
        b.ntiles = (long long)p * L * b.ntz;
        b.in_hi = Nx * L * M; b.in_lo = M; b.in_rq = 0; b.in_rl = L * M;
        b.out_hi = Nx * L * (M + 1); b.out_lo = M + 1; b.out_rq = 0; b.out_rl = L * (M + 1);
        rc = launch(kx->s_fn[0][KIND_LIN_LIN], b.ntiles, pl->grid_x[0], kx->s_threads, kx->s_smem, &b, st);
    }
    rec.mark(slot++);
    return rc;
}

// I1 (step 5 reversed): x-axis inverse FFT inside each of the qn virtual slabs: spectrum (pitch M+1, its
// column 0 replaced by the packed `side` [qn][Nx][L]) -> slab (pitch M).
static int stage_inv_x(const fft3d_plan_t* pl, const void* d_in, const void* side, void* slab, cudaStream_t st,
                       Recorder& rec, int& slot) {
    const long long Nx = pl->Nx, M = pl->M, L = pl->L, p = pl->qn;
    const KernelSet* kx = pl->kx;
    int rc;
    if (x_impl(pl, 1) != IMPL_PLAIN) {
        TensorMapBlob mi, mo;
        TensorMapBlob mi2;
        const int tc = kx->tma_tc_x, of = kx->tma_oddfix;
        if (!map_user_x(pl, &mi, d_in, tc, pl->x_rows) || !map_user_x(pl, &mi2, d_in, tc + 2, pl->x_rows) ||
            !map_slab_x(pl, &mo, slab, tc, pl->x_rows)) return FFT3D_ECUDA;
        TmaArgs ta{};
        ta.tw = pl->tw_x; ta.ntz = (int)(M / tc);
        ta.ntiles = of ? (long long)p * (L / 2) * (2 * ta.ntz) : (long long)p * L * ta.ntz;
        ta.L = (int)L; ta.Nx = (int)Nx; ta.Mp1 = (int)(M + 1); ta.in_rows = pl->x_rows; ta.out_rows = pl->x_rows;
        if (x_impl(pl, 1) == IMPL_TMA_SPLIT4) rc = launch_x_split4(pl, 1, d_in, slab, st);
        else if (x_impl(pl, 1) == IMPL_TMA_SPLIT2) rc = launch_x_split2(pl, 1, d_in, slab, st);
        else rc = launch_tma(kx->tma_fn[TMA_X_INV], kx->tma_threads_x, kx->tma_smem_x, pl->num_sms, mi, mi2, mo, ta, st);
        rec.mark(slot++);
        // packed column 0 of the result: x-transform of the side buffer, written over the (meaningless)
        // column the tiles produced from the user's raw kz = 0 plane
        if (rc == FFT3D_OK) {
            StridedArgs c0{};
            c0.in = side; c0.out = slab; c0.col0 = nullptr; c0.tw = pl->tw_x;
            c0.ntz = (int)((L + kx->tc - 1) / kx->tc); c0.ncols = (int)L; c0.a_lo = 1; c0.L = (int)Nx;
            c0.ntiles = (long long)p * c0.ntz;
            c0.in_hi = Nx * L; c0.in_lo = 0; c0.in_rq = 0; c0.in_rl = L;
            c0.out_hi = Nx * L * M; c0.out_lo = 0; c0.out_rq = 0; c0.out_rl = L * M; c0.out_cs = M;
            rc = launch(kx->s_fn[1][KIND_LIN_LIN], c0.ntiles, pl->grid_x[1], kx->s_threads, kx->s_smem, &c0, st);
        }
    } else {
        StridedArgs b{};
        b.in = d_in; b.out = slab; b.col0 = side; b.tw = pl->tw_x;
        b.ntz = (int)((M + kx->tc - 1) / kx->tc); b.ncols = (int)M; b.a_lo = (int)L; b.L = (int)Nx;
        b.ntiles = (long long)p * L * b.ntz;
        b.in_hi = Nx * L * (M + 1); b.in_lo = M + 1; b.in_rq = 0; b.in_rl = L * (M + 1);
        b.c0_hi = Nx * L; b.c0_lo = 1; b.c0_rl = L;
        b.out_hi = Nx * L * M; b.out_lo = M; b.out_rq = 0; b.out_rl = L * M;
        rc = launch(kx->s_fn[1][KIND_LIN_LIN], b.ntiles, pl->grid_x[1], kx->s_threads, kx->s_smem, &b, st);
    }
    rec.mark(slot++);
    return rc;
}

// I2 + I3 (steps 4..1 reversed, with the 1/(NxNyNz) normalisation) of planes [xp0, xp0 + xpn):
// slab array -> real `d_out`.  Fused: through `ring`; unfused: through `scratch` [xpn][Ny][M].
static int stage_inv_yz(const fft3d_plan_t* pl, const void* slab, void* scratch, void* d_out, void* ring, unsigned* flags,
                        cudaStream_t st, Recorder& rec, int& slot) {
    const long long Nxp = pl->xpn, Ny = pl->Ny, M = pl->M, L = pl->L;
    int rc;
    if (use_fused(pl)) {
        rc = launch_fused(pl, 1, nullptr, d_out, const_cast<void*>(slab), ring, flags, st);
        rec.mark(slot++);
        return rc;
    }
    // I2: y-axis inverse FFT gathering rows from the slab layout: slab -> scratch [x][y][M]
    const KernelSet* ky = pl->ky;
    if (y_impl(pl) == IMPL_TMA_SPLIT2) {
        rc = launch_y_split2(pl, 1, slab, scratch, st);
    } else if (y_impl(pl) == IMPL_TMA) {
        TensorMapBlob mi, mo;
        if (!map_slab_y(pl, &mi, slab, ky->tma_tc, pl->y_rows_slab) ||
            !map_natural(pl, &mo, scratch, ky->tma_tc, pl->y_rows_nat)) return FFT3D_ECUDA;
        TmaArgs ta{};
        ta.tw = pl->tw_y; ta.ntz = (int)(M / ky->tma_tc); ta.ntiles = Nxp * ta.ntz;
        ta.L = (int)L; ta.Nx = (int)pl->Nx; ta.Mp1 = (int)(M + 1); ta.in_rows = pl->y_rows_slab; ta.out_rows = pl->y_rows_nat;
        rc = launch_tma(ky->tma_fn[TMA_Y_INV], ky->tma_threads, ky->tma_smem_y, pl->num_sms, mi, mi, mo, ta, st);
    } else {
        StridedArgs a{};
        a.in = reinterpret_cast<const unsigned char*>(slab) + (size_t)pl->xp0 * L * M * 2 * pl->esize;
        a.out = scratch; a.col0 = nullptr; a.tw = pl->tw_y;
        a.ntz = (int)((M + ky->tc - 1) / ky->tc); a.ncols = (int)M; a.a_lo = 1; a.L = (int)L;
        a.ntiles = Nxp * a.ntz;
        a.in_hi = L * M; a.in_lo = 0; a.in_rq = pl->sNx * L * M; a.in_rl = M;
        a.out_hi = Ny * pl->nat_pitch; a.out_lo = 0; a.out_rq = 0; a.out_rl = pl->nat_pitch;
        rc = launch(ky->s_fn[1][KIND_SLAB_LIN], a.ntiles, pl->grid_y[1], ky->s_threads, ky->s_smem, &a, st);
    }
    if (rc != FFT3D_OK) return rc;
    rec.mark(slot++);

    // I3: z-axis C2R with the 1/(NxNyNz) normalisation: scratch -> d_out
    const KernelSet* kz = pl->kz;
    ZArgs z{};
    z.in = scratch; z.out = d_out; z.tw = pl->tw_z; z.twz = pl->twz; z.nrows = Nxp * Ny;
    z.in_pitch = z.out_pitch = pl->nat_pitch;
    z.scale = 1.0 / ((double)pl->Nx * (double)Ny * (double)pl->Nz);
    if (z_impl(pl) == IMPL_BULK) rc = launch_zbulk(pl, 1, scratch, d_out, z.scale, st);
    else rc = launch(kz->z_fn[1], (z.nrows + kz->z_rpb - 1) / kz->z_rpb, pl->grid_z[1], kz->z_threads, kz->z_smem, &z, st);
    rec.mark(slot++);
    return rc;
}

// where a plain plan keeps the pieces of its fused pipeline in the workspace: [slab array | ring | side | flags]
static void* ws_ring(const fft3d_plan_t* pl, void* d_work) { return reinterpret_cast<unsigned char*>(d_work) + pl->slab_bytes; }
static void* ws_side(const fft3d_plan_t* pl, void* d_work) { return reinterpret_cast<unsigned char*>(d_work) + pl->slab_bytes + pl->ring_bytes; }
static unsigned* ws_flags(const fft3d_plan_t* pl, void* d_work) {
    return reinterpret_cast<unsigned*>(reinterpret_cast<unsigned char*>(d_work) + pl->slab_bytes + pl->ring_bytes + pl->side_bytes);
}

static void* pencil_staging(const fft3d_plan_t* pl, void* d_work) {
    const size_t base = pl->slab_bytes + pl->ring_bytes + pl->side_bytes + pl->flags_bytes;
    return reinterpret_cast<unsigned char*>(d_work) + ((base + 255) & ~(size_t)255);
}
static int pencil_convert(const fft3d_plan_t* pl, const void* src, void* dst, int dir, cudaStream_t st) {
    PencilArgs a{};
    a.src = src; a.dst = dst; a.rows_per_a = pl->Nx * pl->L; a.nrows = (long long)pl->p * a.rows_per_a;
    a.M = (int)pl->M; a.py = pl->pencil_py; a.dir = dir;
    if (launch_pencil_convert(pl->dtype, a, st) != cudaSuccess) { cudaGetLastError(); return FFT3D_ECUDA; }
    return FFT3D_OK;
}

int fft3d_r2c(const fft3d_plan_t* pl, const void* d_in, void* d_out, void* d_work, void* stream) {
    if (pl == nullptr || pl->kind != 0 || pl->dist_G != 0 || pl->inplace || d_in == nullptr || d_out == nullptr || d_work == nullptr) return FFT3D_EINVAL;
    if (wrong_device(pl)) return FFT3D_EINVAL;          // the current device is not the plan's
    const size_t rb = fft3d_real_bytes(pl), cb = fft3d_complex_bytes(pl), wb = fft3d_workspace_bytes(pl);
    if (((uintptr_t)d_in | (uintptr_t)d_out | (uintptr_t)d_work) & 15) return FFT3D_EINVAL;
    if (overlap(d_in, rb, d_out, cb) || overlap(d_in, rb, d_work, wb) || overlap(d_out, cb, d_work, wb))
        return FFT3D_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    Recorder rec(pl, 0, st);
    int slot = 0;
    rec.mark(slot++);
    // pencil-layout plans: the slab-layout spectrum (p = px) is staged behind the workspace and cut into the py
    // column ranges of the rank grid by one more pass
    void* user_out = d_out;
    if (pl->pencil_py > 0) d_out = pencil_staging(pl, d_work);
    // fused: real -> (ring in L2) -> slab array in the workspace; unfused: real -> d_out (scratch use) -> workspace
    int rc = stage_fwd_zy(pl, d_in, d_out, d_work, ws_ring(pl, d_work), ws_flags(pl, d_work), st, rec, slot);
    if (rc != FFT3D_OK) return rc;
    rc = stage_fwd_x(pl, d_work, d_out, st, rec, slot);
    if (rc != FFT3D_OK) return rc;
    // column 0 holds A + iB (planes kz = 0 and kz = Nz/2): separate them in place
    PlaneArgs f{};
    f.src = nullptr; f.dst = d_out; f.Nx = (int)pl->Nx; f.Ny = (int)pl->Ny; f.L = (int)pl->L; f.M = (int)pl->M;
    if (launch_unpack_nyquist(pl->dtype, f, st) != cudaSuccess) { cudaGetLastError(); return FFT3D_ECUDA; }
    rec.mark(slot++);
    if (pl->pencil_py > 0) {
        if (pencil_convert(pl, d_out, user_out, 0, st) != FFT3D_OK) return FFT3D_ECUDA;
        rec.mark(slot++);
    }
    return FFT3D_OK;
}

int fft3d_c2r(const fft3d_plan_t* pl, const void* d_in, void* d_out, void* d_work, void* stream) {
    if (pl == nullptr || pl->kind != 0 || pl->dist_G != 0 || pl->inplace || d_in == nullptr || d_out == nullptr || d_work == nullptr) return FFT3D_EINVAL;
    if (wrong_device(pl)) return FFT3D_EINVAL;          // the current device is not the plan's
    const size_t rb = fft3d_real_bytes(pl), cb = fft3d_complex_bytes(pl), wb = fft3d_workspace_bytes(pl);
    if (((uintptr_t)d_in | (uintptr_t)d_out | (uintptr_t)d_work) & 15) return FFT3D_EINVAL;
    if (overlap(d_in, cb, d_out, rb) || overlap(d_in, cb, d_work, wb) || overlap(d_out, rb, d_work, wb))
        return FFT3D_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    Recorder rec(pl, 1, st);
    int slot = 0;
    rec.mark(slot++);
    if (pl->pencil_py > 0) {                       // pencil blocks -> slab rows in the staging area, then as usual
        void* staged = pencil_staging(pl, d_work);
        if (pencil_convert(pl, d_in, staged, 1, st) != FFT3D_OK) return FFT3D_ECUDA;
        rec.mark(slot++);
        d_in = staged;
    }
    const bool fz = use_fused(pl);
    // pre-pack: side[q][kx][ky_l] = sym(plane kz=0) + i sym(plane kz=Nz/2) (reading R8: only the Hermitian part of
    // the two self-conjugate planes enters Eq. (2)+(3)).  Fused: I1 writes the slab array in the workspace and I2+I3
    // go from there to d_out, so the side buffer sits behind the ring; unfused: the side buffer sits at the start
    // of the workspace until I1 has consumed it, I1 -> d_out (scratch use) -> I2 -> workspace -> I3 -> d_out.
    void* side = fz ? ws_side(pl, d_work) : d_work;
    void* slab = fz ? d_work : d_out;
    PlaneArgs f{};
    f.src = d_in; f.dst = side; f.Nx = (int)pl->Nx; f.Ny = (int)pl->Ny; f.L = (int)pl->L; f.M = (int)pl->M;
    if (launch_pack_nyquist(pl->dtype, f, st) != cudaSuccess) { cudaGetLastError(); return FFT3D_ECUDA; }
    rec.mark(slot++);
    int rc = stage_inv_x(pl, d_in, side, slab, st, rec, slot);
    if (rc != FFT3D_OK) return rc;
    return stage_inv_yz(pl, slab, d_work, d_out, ws_ring(pl, d_work), ws_flags(pl, d_work), st, rec, slot);
}

// ---------------------------------------------------------------------------------------------------------
// Padded in-place layout ("each GPU now contains Nx/p x Ny x (Nz/2+1) data points", i.e.
// FFTW-style rows of 2*(Nz/2+1) reals): the real field and its half spectrum share ONE buffer, with the single
// workspace beside it.  Rows of Nz/2+1 fp32 complex start on 8-byte boundaries, which neither bulk copies
// nor tensor maps can address, so the passes that touch this layout -- z (in place, row by row) and the natural
// side of y -- run the plain-load kernels; the x pass and the slab side keep the TMA kernels.
//   forward : z R2C in place (pitch M+1) -> y C2C: data -> slab array in the workspace -> x C2C: workspace -> data
//   inverse : x C2C: data -> workspace -> y C2C: workspace -> data (pitch M+1) -> z C2R in place
// ---------------------------------------------------------------------------------------------------------
int fft3d_plan_inplace(fft3d_plan_t** out, long long Nx, long long Ny, long long Nz, int dtype, int virtual_slabs) {
    int rc = plan_create(out, Nx, Ny, Nz, dtype, virtual_slabs, 0);
    if (rc != FFT3D_OK) return rc;
    fft3d_plan_t* pl = *out;
    pl->inplace = 1;
    pl->nat_pitch = pl->M + 1;
    pl->fused = pl->fused_default = false;
    pl->ring_bytes = 0;
    pl->flags_bytes = 0;
    pl->side_bytes = ((size_t)Nx * Ny * 2 * pl->esize + 255) & ~(size_t)255;      // packed column of the inverse
    return FFT3D_OK;
}

int fft3d_r2c_inplace(const fft3d_plan_t* pl, void* d_data, void* d_work, void* stream) {
    if (pl == nullptr || !pl->inplace || d_data == nullptr || d_work == nullptr) return FFT3D_EINVAL;
    if (wrong_device(pl)) return FFT3D_EINVAL;          // the current device is not the plan's
    if (((uintptr_t)d_data | (uintptr_t)d_work) & 15) return FFT3D_EINVAL;
    if (overlap(d_data, fft3d_complex_bytes(pl), d_work, fft3d_workspace_bytes(pl))) return FFT3D_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    Recorder rec(pl, 0, st);
    int slot = 0;
    rec.mark(slot++);
    int rc = stage_fwd_zy(pl, d_data, d_data, d_work, nullptr, nullptr, st, rec, slot);
    if (rc != FFT3D_OK) return rc;
    rc = stage_fwd_x(pl, d_work, d_data, st, rec, slot);
    if (rc != FFT3D_OK) return rc;
    PlaneArgs f{};
    f.src = nullptr; f.dst = d_data; f.Nx = (int)pl->Nx; f.Ny = (int)pl->Ny; f.L = (int)pl->L; f.M = (int)pl->M;
    if (launch_unpack_nyquist(pl->dtype, f, st) != cudaSuccess) { cudaGetLastError(); return FFT3D_ECUDA; }
    rec.mark(slot++);
    return FFT3D_OK;
}

int fft3d_c2r_inplace(const fft3d_plan_t* pl, void* d_data, void* d_work, void* stream) {
    if (pl == nullptr || !pl->inplace || d_data == nullptr || d_work == nullptr) return FFT3D_EINVAL;
    if (wrong_device(pl)) return FFT3D_EINVAL;          // the current device is not the plan's
    if (((uintptr_t)d_data | (uintptr_t)d_work) & 15) return FFT3D_EINVAL;
    if (overlap(d_data, fft3d_complex_bytes(pl), d_work, fft3d_workspace_bytes(pl))) return FFT3D_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    Recorder rec(pl, 1, st);
    int slot = 0;
    rec.mark(slot++);
    void* side = reinterpret_cast<unsigned char*>(d_work) + pl->slab_bytes;       // behind the slab array
    PlaneArgs f{};
    f.src = d_data; f.dst = side; f.Nx = (int)pl->Nx; f.Ny = (int)pl->Ny; f.L = (int)pl->L; f.M = (int)pl->M;
    if (launch_pack_nyquist(pl->dtype, f, st) != cudaSuccess) { cudaGetLastError(); return FFT3D_ECUDA; }
    rec.mark(slot++);
    int rc = stage_inv_x(pl, d_data, side, d_work, st, rec, slot);
    if (rc != FFT3D_OK) return rc;
    return stage_inv_yz(pl, d_work, d_data, d_data, nullptr, nullptr, st, rec, slot);
}

// ---------------------------------------------------------------------------------------------------------
// Distributed slab decomposition over G GPUs: the paper's method itself.
// Rank r owns the x-slab [Nx/G][Ny][Nz] of the real field and the y-slab [Nx][Ny/G][Nz/2+1] of the spectrum.
// The stages below run the SAME launch code as the single-GPU transform on a copy of the plan narrowed to the
// rank's planes / virtual slab; what differs between the exchange back-ends is only where the slab array lives.
// ---------------------------------------------------------------------------------------------------------
static size_t dist_scratch_bytes(const fft3d_plan_t* pl) { return pl->slab_bytes / (size_t)pl->dist_G; }
static size_t dist_side_bytes(const fft3d_plan_t* pl) { return (((size_t)pl->Nx * pl->L * 2 * pl->esize) + 255) & ~(size_t)255; }
static unsigned char* dist_ring(const fft3d_plan_t* pl, void* w) { return reinterpret_cast<unsigned char*>(w) + dist_scratch_bytes(pl); }
static unsigned char* dist_side(const fft3d_plan_t* pl, void* w) { return dist_ring(pl, w) + pl->ring_bytes; }
static unsigned* dist_flags(const fft3d_plan_t* pl, void* w) { return reinterpret_cast<unsigned*>(dist_side(pl, w) + dist_side_bytes(pl)); }

int fft3d_plan_dist(fft3d_plan_t** out, long long Nx, long long Ny, long long Nz, int dtype, int G, int rank) {
    if (out == nullptr) return FFT3D_EINVAL;
    *out = nullptr;
    if (G < 1 || G > 16 || rank < 0 || rank >= G) return FFT3D_EINVAL;
    int rc = plan_create(out, Nx, Ny, Nz, dtype, G, 0);              // p = G: checks G | Nx and G | Ny
    if (rc != FFT3D_OK) return rc;
    fft3d_plan_t* pl = *out;
    pl->dist_G = G; pl->dist_rank = rank;
    const long long Nxl = Nx / G;
    // plan_create judged the bulk-pipelined z kernel on the rows of the WHOLE grid; the stages run it on the local slab's
    // (Nx/G)*Ny rows, which must be whole tiles too (otherwise: plain-load z kernel, and no fused z+y pass, which needs it)
    if (pl->bulk_z && (Nxl * Ny) % pl->kz->zb_rpt != 0) {
        pl->bulk_z = false;
        pl->fused = pl->fused_default = false;
    }
    if (pl->fused) {
        // the ring holds planes of the local x-slab only; fusion pays once the LOCAL arrays are far larger than L2
        if (Nxl < 2) pl->fused = pl->fused_default = false;
        else if (pl->fz_R > Nxl) {
            pl->fz_R = pl->fz_R_max = (int)Nxl;
            pl->ring_bytes = (size_t)Ny * pl->M * 2 * pl->esize * (size_t)Nxl;
        }
        pl->fused_default = pl->fused_default && dist_scratch_bytes(pl) >= ((size_t)2 << 30);
    }
    if (!pl->fused) {       // size the (unused) fused pieces of the workspace for the flags only
        pl->ring_bytes = 0;
        pl->flags_bytes = 256;
    }
    return FFT3D_OK;
}

size_t fft3d_dist_bytes(const fft3d_plan_t* pl, int which) {
    if (pl == nullptr || pl->dist_G == 0) return 0;
    const size_t G = (size_t)pl->dist_G, csz = 2 * (size_t)pl->esize;
    switch (which) {
        case FFT3D_DIST_REAL: return (size_t)pl->Nx * pl->Ny * pl->Nz * pl->esize / G;
        case FFT3D_DIST_SLAB: return pl->slab_bytes / G;
        case FFT3D_DIST_SPEC: return (size_t)pl->Nx * pl->L * (pl->M + 1) * csz;
        case FFT3D_DIST_PLANES: return 2 * (size_t)pl->Nx * pl->L * csz;
        case FFT3D_DIST_WORK: return dist_scratch_bytes(pl) + pl->ring_bytes + dist_side_bytes(pl) + pl->flags_bytes;
        default: return 0;
    }
}

// the plan narrowed to this rank's planes of the z and y passes
static int dist_view_zy(const fft3d_plan_t* pl, int layout, fft3d_plan_t* v) {
    if (layout != FFT3D_XCHG_UNIFIED && layout != FFT3D_XCHG_CHUNKS) return FFT3D_EINVAL;
    *v = *pl;
    v->timing = nullptr;
    v->xpn = pl->Nx / pl->dist_G;
    if (layout == FFT3D_XCHG_UNIFIED) { v->xp0 = pl->dist_rank * v->xpn; v->sNx = pl->Nx; }   // [G][Nx][L][M], part q on rank q
    else { v->xp0 = 0; v->sNx = v->xpn; }                                                       // [G][Nx/G][L][M], all local
    return FFT3D_OK;
}

int fft3d_dist_fwd_local(const fft3d_plan_t* pl, const void* d_real_slab, void* d_xchg, int layout, void* d_work, void* stream) {
    if (pl == nullptr || pl->dist_G == 0 || d_real_slab == nullptr || d_xchg == nullptr || d_work == nullptr) return FFT3D_EINVAL;
    if (wrong_device(pl)) return FFT3D_EINVAL;          // the current device is not the plan's
    if (((uintptr_t)d_real_slab | (uintptr_t)d_xchg | (uintptr_t)d_work) & 15) return FFT3D_EINVAL;
    fft3d_plan_t v;
    int rc = dist_view_zy(pl, layout, &v);
    if (rc != FFT3D_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    Recorder rec(&v, 0, st);
    int slot = 0;
    return stage_fwd_zy(&v, d_real_slab, d_work, d_xchg, dist_ring(pl, d_work), dist_flags(pl, d_work), st, rec, slot);
}

int fft3d_dist_fwd_x(const fft3d_plan_t* pl, const void* d_slab_part, void* d_spec_part, void* stream) {
    if (pl == nullptr || pl->dist_G == 0 || d_slab_part == nullptr || d_spec_part == nullptr) return FFT3D_EINVAL;
    if (wrong_device(pl)) return FFT3D_EINVAL;          // the current device is not the plan's
    if (((uintptr_t)d_slab_part | (uintptr_t)d_spec_part) & 15) return FFT3D_EINVAL;
    fft3d_plan_t v = *pl;
    v.timing = nullptr;
    v.qn = 1;
    cudaStream_t st = (cudaStream_t)stream;
    Recorder rec(&v, 0, st);
    int slot = 0;
    return stage_fwd_x(&v, d_slab_part, d_spec_part, st, rec, slot);
}

static int dist_planes(const fft3d_plan_t* pl, const void* d_spec_part, void* d_plane_part, int ncols, void* stream) {
    if (pl == nullptr || pl->dist_G == 0 || d_spec_part == nullptr || d_plane_part == nullptr) return FFT3D_EINVAL;
    if (wrong_device(pl)) return FFT3D_EINVAL;          // the current device is not the plan's
    if (((uintptr_t)d_spec_part | (uintptr_t)d_plane_part) & 15) return FFT3D_EINVAL;
    DistPlaneArgs a{};
    a.spec = d_spec_part; a.own = d_plane_part;
    a.Nx = (int)pl->Nx; a.Ny = (int)pl->Ny; a.L = (int)pl->L; a.M = (int)pl->M; a.q = pl->dist_rank; a.ncols = ncols;
    if (launch_dist_extract(pl->dtype, a, (cudaStream_t)stream) != cudaSuccess) { cudaGetLastError(); return FFT3D_ECUDA; }
    return FFT3D_OK;
}
int fft3d_dist_fwd_col0(const fft3d_plan_t* pl, const void* d_spec_part, void* d_plane_part, void* stream) {
    return dist_planes(pl, d_spec_part, d_plane_part, 1, stream);
}
int fft3d_dist_inv_planes(const fft3d_plan_t* pl, const void* d_spec_part, void* d_plane_part, void* stream) {
    return dist_planes(pl, d_spec_part, d_plane_part, 2, stream);
}

int fft3d_dist_fwd_unpack(const fft3d_plan_t* pl, void* d_spec_part, const void* const* d_plane_parts, void* stream) {
    if (pl == nullptr || pl->dist_G == 0 || d_spec_part == nullptr || d_plane_parts == nullptr) return FFT3D_EINVAL;
    if (wrong_device(pl)) return FFT3D_EINVAL;          // the current device is not the plan's
    if ((uintptr_t)d_spec_part & 15) return FFT3D_EINVAL;
    DistPlaneArgs a{};
    a.spec_out = d_spec_part;
    for (int q = 0; q < pl->dist_G; ++q) { if (d_plane_parts[q] == nullptr) return FFT3D_EINVAL; a.parts[q] = d_plane_parts[q]; }
    a.Nx = (int)pl->Nx; a.Ny = (int)pl->Ny; a.L = (int)pl->L; a.M = (int)pl->M; a.q = pl->dist_rank; a.ncols = 1;
    if (launch_dist_unpack(pl->dtype, a, (cudaStream_t)stream) != cudaSuccess) { cudaGetLastError(); return FFT3D_ECUDA; }
    return FFT3D_OK;
}

int fft3d_dist_inv_pack(const fft3d_plan_t* pl, const void* const* d_plane_parts, void* d_work, void* stream) {
    if (pl == nullptr || pl->dist_G == 0 || d_plane_parts == nullptr || d_work == nullptr) return FFT3D_EINVAL;
    if (wrong_device(pl)) return FFT3D_EINVAL;          // the current device is not the plan's
    DistPlaneArgs a{};
    a.side = dist_side(pl, d_work);
    for (int q = 0; q < pl->dist_G; ++q) { if (d_plane_parts[q] == nullptr) return FFT3D_EINVAL; a.parts[q] = d_plane_parts[q]; }
    a.Nx = (int)pl->Nx; a.Ny = (int)pl->Ny; a.L = (int)pl->L; a.M = (int)pl->M; a.q = pl->dist_rank; a.ncols = 1;
    if (launch_dist_pack(pl->dtype, a, (cudaStream_t)stream) != cudaSuccess) { cudaGetLastError(); return FFT3D_ECUDA; }
    return FFT3D_OK;
}

int fft3d_dist_inv_x(const fft3d_plan_t* pl, const void* d_spec_part, void* d_slab_part, void* d_work, void* stream) {
    if (pl == nullptr || pl->dist_G == 0 || d_spec_part == nullptr || d_slab_part == nullptr || d_work == nullptr) return FFT3D_EINVAL;
    if (wrong_device(pl)) return FFT3D_EINVAL;          // the current device is not the plan's
    if (((uintptr_t)d_slab_part | (uintptr_t)d_spec_part | (uintptr_t)d_work) & 15) return FFT3D_EINVAL;
    fft3d_plan_t v = *pl;
    v.timing = nullptr;
    v.qn = 1;
    cudaStream_t st = (cudaStream_t)stream;
    Recorder rec(&v, 1, st);
    int slot = 0;
    return stage_inv_x(&v, d_spec_part, dist_side(pl, d_work), d_slab_part, st, rec, slot);
}

int fft3d_dist_inv_local(const fft3d_plan_t* pl, const void* d_xchg, int layout, void* d_real_slab, void* d_work, void* stream) {
    if (pl == nullptr || pl->dist_G == 0 || d_real_slab == nullptr || d_xchg == nullptr || d_work == nullptr) return FFT3D_EINVAL;
    if (wrong_device(pl)) return FFT3D_EINVAL;          // the current device is not the plan's
    if (((uintptr_t)d_real_slab | (uintptr_t)d_xchg | (uintptr_t)d_work) & 15) return FFT3D_EINVAL;
    fft3d_plan_t v;
    int rc = dist_view_zy(pl, layout, &v);
    if (rc != FFT3D_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    Recorder rec(&v, 1, st);
    int slot = 0;
    return stage_inv_yz(&v, d_xchg, d_work, d_real_slab, dist_ring(pl, d_work), dist_flags(pl, d_work), st, rec, slot);
}

// 3D C2C (the paper's R2C, C2C and C2R share one workspace).  direction -1: forward,
// unnormalised (z rows, y lines with the slab permutation of steps 2-4, x lines: steps 1 and 5);
// +1: inverse, scaled by 1/(NxNyNz), the passes in reverse order.
int fft3d_c2c(const fft3d_plan_t* pl, const void* d_in, void* d_out, void* d_work, int direction, void* stream) {
    if (pl == nullptr || pl->kind != 1 || d_in == nullptr || d_out == nullptr || d_work == nullptr) return FFT3D_EINVAL;
    if (wrong_device(pl)) return FFT3D_EINVAL;          // the current device is not the plan's
    if (direction != -1 && direction != 1) return FFT3D_EINVAL;
    const size_t cb = fft3d_complex_bytes(pl), wb = fft3d_workspace_bytes(pl);
    if (((uintptr_t)d_in | (uintptr_t)d_out | (uintptr_t)d_work) & 15) return FFT3D_EINVAL;
    if (overlap(d_in, cb, d_out, cb) || overlap(d_in, cb, d_work, wb) || overlap(d_out, cb, d_work, wb))
        return FFT3D_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    const long long Nx = pl->Nx, Ny = pl->Ny, M = pl->M, L = pl->L, p = pl->p;
    const KernelSet *kz = pl->kz, *ky = pl->ky, *kx = pl->kx;
    const int d = direction < 0 ? 0 : 1;
    Recorder rec(pl, d, st);
    int slot = 0, rc = FFT3D_OK;
    rec.mark(slot++);

    auto z_pass = [&](const void* in, void* out) -> int {
        if (!(use_tma(pl) && pl->bulk_zc)) {            // plain-load rows: any length, any row count
            ZArgs zp{};
            zp.in = in; zp.out = out; zp.tw = pl->tw_z; zp.twz = nullptr; zp.nrows = Nx * Ny;
            zp.scale = 1.0 / ((double)Nx * (double)Ny * (double)pl->Nz);
            return launch(kz->zp_fn[d], (zp.nrows + kz->z_rpb - 1) / kz->z_rpb, pl->grid_zp[d], kz->z_threads, kz->z_smem, &zp, st);
        }
        ZBulkArgs z{};
        z.in = in; z.out = out; z.tw = pl->tw_zc; z.twz = nullptr;
        z.ntiles = Nx * Ny / kz->zc_rpt;
        z.scale = 1.0 / ((double)Nx * (double)Ny * (double)pl->Nz);
        long long g = z.ntiles < pl->num_sms ? z.ntiles : pl->num_sms;
        void* argv[1] = {&z};
        cudaError_t e = cudaLaunchKernel(kz->zc_fn[d], dim3((unsigned)g), dim3((unsigned)kz->zc_threads), argv, kz->zc_smem, st);
        if (e != cudaSuccess) { cudaGetLastError(); return FFT3D_ECUDA; }
        return FFT3D_OK;
    };
    auto y_pass = [&](const void* in, void* out) -> int {       // forward: natural -> slab; inverse: slab -> natural
        if (y_impl(pl) == IMPL_TMA_SPLIT2) return launch_y_split2(pl, d, in, out, st);
        if (y_impl(pl) == IMPL_TMA) {
            TensorMapBlob mi, mo;
            bool ok = d == 0 ? (map_natural(pl, &mi, in, ky->tma_tc, pl->y_rows_nat) && map_slab_y(pl, &mo, out, ky->tma_tc, pl->y_rows_slab))
                             : (map_slab_y(pl, &mi, in, ky->tma_tc, pl->y_rows_slab) && map_natural(pl, &mo, out, ky->tma_tc, pl->y_rows_nat));
            if (!ok) return FFT3D_ECUDA;
            TmaArgs ta{};
            ta.tw = pl->tw_y; ta.ntz = (int)(M / ky->tma_tc); ta.ntiles = Nx * ta.ntz;
            ta.L = (int)L; ta.Nx = (int)Nx; ta.Mp1 = (int)M;
            ta.in_rows = d == 0 ? pl->y_rows_nat : pl->y_rows_slab; ta.out_rows = d == 0 ? pl->y_rows_slab : pl->y_rows_nat;
            return launch_tma(ky->tma_fn[d == 0 ? TMA_Y_FWD : TMA_Y_INV], ky->tma_threads, ky->tma_smem_y, pl->num_sms, mi, mi, mo, ta, st);
        }
        StridedArgs a{};
        a.in = in; a.out = out; a.col0 = nullptr; a.tw = pl->tw_y;
        a.ntz = (int)((M + ky->tc - 1) / ky->tc); a.ncols = (int)M; a.a_lo = 1; a.L = (int)L;
        a.ntiles = Nx * a.ntz;
        if (d == 0) {
            a.in_hi = Ny * M; a.in_lo = 0; a.in_rq = 0; a.in_rl = M;
            a.out_hi = L * M; a.out_lo = 0; a.out_rq = Nx * L * M; a.out_rl = M;
            return launch(ky->s_fn[0][KIND_LIN_SLAB], a.ntiles, pl->grid_y[0], ky->s_threads, ky->s_smem, &a, st);
        }
        a.in_hi = L * M; a.in_lo = 0; a.in_rq = Nx * L * M; a.in_rl = M;
        a.out_hi = Ny * M; a.out_lo = 0; a.out_rq = 0; a.out_rl = M;
        return launch(ky->s_fn[1][KIND_SLAB_LIN], a.ntiles, pl->grid_y[1], ky->s_threads, ky->s_smem, &a, st);
    };
    auto x_pass = [&](const void* in, void* out) -> int {       // lines along x inside every virtual slab, pitch M
        if (x_impl(pl, d) == IMPL_TMA) {
            // X_FWD reads the 4-D slab view and writes the flattened one, X_INV the other way round; with one
            // pitch M on both sides the two views describe the same layout
            TensorMapBlob mi, mo;
            const int tc = kx->tma_tc_x;
            bool ok = d == 0 ? (map_slab_x(pl, &mi, in, tc, pl->x_rows) && map_user_x(pl, &mo, out, tc, pl->x_rows, M))
                             : (map_user_x(pl, &mi, in, tc, pl->x_rows, M) && map_slab_x(pl, &mo, out, tc, pl->x_rows));
            if (!ok) return FFT3D_ECUDA;
            TmaArgs ta{};
            ta.tw = pl->tw_x; ta.ntz = (int)(M / tc); ta.ntiles = (long long)p * L * ta.ntz;
            ta.L = (int)L; ta.Nx = (int)Nx; ta.Mp1 = (int)M; ta.in_rows = pl->x_rows; ta.out_rows = pl->x_rows;
            return launch_tma(kx->xc_fn[d], kx->tma_threads_x, kx->xc_smem, pl->num_sms, mi, mi, mo, ta, st);
        }
        StridedArgs b{};
        b.in = in; b.out = out; b.col0 = nullptr; b.tw = pl->tw_x;
        b.ntz = (int)((M + kx->tc - 1) / kx->tc); b.ncols = (int)M; b.a_lo = (int)L; b.L = (int)Nx;
        b.ntiles = (long long)p * L * b.ntz;
        b.in_hi = Nx * L * M; b.in_lo = M; b.in_rq = 0; b.in_rl = L * M;
        b.out_hi = Nx * L * M; b.out_lo = M; b.out_rq = 0; b.out_rl = L * M;
        return launch(kx->s_fn[d][KIND_LIN_LIN], b.ntiles, pl->grid_x[d], kx->s_threads, kx->s_smem, &b, st);
    };

    if (use_fused(pl)) {
        if (d == 0) {
            rc = launch_fused(pl, 0, d_in, nullptr, d_work, ws_ring(pl, d_work), ws_flags(pl, d_work), st);   rec.mark(slot++); if (rc != FFT3D_OK) return rc;
            rc = x_pass(d_work, d_out);                                    rec.mark(slot++);
        } else {
            rc = x_pass(d_in, d_work);                                     rec.mark(slot++); if (rc != FFT3D_OK) return rc;
            rc = launch_fused(pl, 1, nullptr, d_out, d_work, ws_ring(pl, d_work), ws_flags(pl, d_work), st);  rec.mark(slot++);
        }
        return rc;
    }
    if (d == 0) {
        rc = z_pass(d_in, d_out);           rec.mark(slot++); if (rc != FFT3D_OK) return rc;
        rc = y_pass(d_out, d_work);         rec.mark(slot++); if (rc != FFT3D_OK) return rc;
        rc = x_pass(d_work, d_out);         rec.mark(slot++);
    } else {
        rc = x_pass(d_in, d_out);           rec.mark(slot++); if (rc != FFT3D_OK) return rc;
        rc = y_pass(d_out, d_work);         rec.mark(slot++); if (rc != FFT3D_OK) return rc;
        rc = z_pass(d_work, d_out);         rec.mark(slot++);
    }
    return rc;
}

static void timing_free(fft3d_plan_t* pl) {
    if (pl->timing == nullptr) return;
    for (int w = 0; w < 2; ++w)
        for (cudaEvent_t e : pl->timing->ev[w]) cudaEventDestroy(e);
    delete pl->timing;
    pl->timing = nullptr;
}

int fft3d_timing_enable(fft3d_plan_t* pl, int max_calls) {
    if (pl == nullptr || pl->dist_G != 0 || max_calls < 0 || max_calls > 4096) return FFT3D_EINVAL;
    timing_free(pl);
    if (max_calls == 0) return FFT3D_OK;
    TimingState* t = new (std::nothrow) TimingState();
    if (t == nullptr) return FFT3D_ENOMEM;
    t->max_calls = max_calls;
    t->calls[0] = t->calls[1] = 0;
    for (int w = 0; w < 2; ++w) {
        t->ev[w].resize((size_t)max_calls * (FFT3D_MAX_LAUNCHES + 1));
        for (auto& e : t->ev[w])
            if (cudaEventCreate(&e) != cudaSuccess) { cudaGetLastError(); pl->timing = t; timing_free(pl); return FFT3D_ECUDA; }
    }
    pl->timing = t;
    return FFT3D_OK;
}

int fft3d_timing_read(fft3d_plan_t* pl, int which, float* ms_sum, int* calls) {
    if (pl == nullptr || pl->timing == nullptr || which < 0 || which > 1 || ms_sum == nullptr || calls == nullptr)
        return FFT3D_EINVAL;
    TimingState* t = pl->timing;
    const int nl = fft3d_launches(pl, which);
    for (int i = 0; i < FFT3D_MAX_LAUNCHES; ++i) ms_sum[i] = 0.f;
    for (int c = 0; c < t->calls[which]; ++c) {
        cudaEvent_t* e = &t->ev[which][(size_t)c * (FFT3D_MAX_LAUNCHES + 1)];
        if (cudaEventSynchronize(e[nl]) != cudaSuccess) { cudaGetLastError(); return FFT3D_ECUDA; }
        for (int i = 0; i < nl; ++i) {
            float ms = 0.f;
            if (cudaEventElapsedTime(&ms, e[i], e[i + 1]) != cudaSuccess) { cudaGetLastError(); return FFT3D_ECUDA; }
            ms_sum[i] += ms;
        }
    }
    *calls = t->calls[which];
    t->calls[which] = 0;
    return FFT3D_OK;
}

static int ensure_host_buffers(fft3d_plan_t* pl) {
    if (pl->h_real != nullptr) return FFT3D_OK;
    if (pl->h_stream == nullptr && cudaStreamCreateWithFlags(&pl->h_stream, cudaStreamNonBlocking) != cudaSuccess) {
        cudaGetLastError();
        pl->h_stream = nullptr;
        return FFT3D_ECUDA;
    }
    if (cudaMalloc(&pl->h_real, pl->kind == 0 ? fft3d_real_bytes(pl) : fft3d_complex_bytes(pl)) != cudaSuccess ||
        cudaMalloc(&pl->h_cplx, fft3d_complex_bytes(pl)) != cudaSuccess ||
        cudaMalloc(&pl->h_work, fft3d_workspace_bytes(pl)) != cudaSuccess) {
        cudaGetLastError();
        cudaFree(pl->h_real); cudaFree(pl->h_cplx); cudaFree(pl->h_work);
        pl->h_real = pl->h_cplx = pl->h_work = nullptr;
        return FFT3D_ENOMEM;
    }
    return FFT3D_OK;
}

int fft3d_r2c_host(fft3d_plan_t* pl, const void* h_in, void* h_out) {
    // in-place and distributed plans have no host-buffer form: refuse them before any device buffer is allocated
    if (pl == nullptr || pl->kind != 0 || pl->inplace || pl->dist_G != 0 || h_in == nullptr || h_out == nullptr) return FFT3D_EINVAL;
    if (wrong_device(pl)) return FFT3D_EINVAL;          // the current device is not the plan's
    int rc = ensure_host_buffers(pl);
    if (rc != FFT3D_OK) return rc;
    cudaStream_t st = pl->h_stream;
    if (cudaMemcpyAsync(pl->h_real, h_in, fft3d_real_bytes(pl), cudaMemcpyHostToDevice, st) != cudaSuccess) {
        cudaGetLastError();
        return FFT3D_ECUDA;
    }
    rc = fft3d_r2c(pl, pl->h_real, pl->h_cplx, pl->h_work, st);
    if (rc != FFT3D_OK) return rc;
    if (cudaMemcpyAsync(h_out, pl->h_cplx, fft3d_complex_bytes(pl), cudaMemcpyDeviceToHost, st) != cudaSuccess ||
        cudaStreamSynchronize(st) != cudaSuccess) {
        cudaGetLastError();
        return FFT3D_ECUDA;
    }
    return FFT3D_OK;
}

int fft3d_c2r_host(fft3d_plan_t* pl, const void* h_in, void* h_out) {
    // in-place and distributed plans have no host-buffer form: refuse them before any device buffer is allocated
    if (pl == nullptr || pl->kind != 0 || pl->inplace || pl->dist_G != 0 || h_in == nullptr || h_out == nullptr) return FFT3D_EINVAL;
    if (wrong_device(pl)) return FFT3D_EINVAL;          // the current device is not the plan's
    int rc = ensure_host_buffers(pl);
    if (rc != FFT3D_OK) return rc;
    cudaStream_t st = pl->h_stream;
    if (cudaMemcpyAsync(pl->h_cplx, h_in, fft3d_complex_bytes(pl), cudaMemcpyHostToDevice, st) != cudaSuccess) {
        cudaGetLastError();
        return FFT3D_ECUDA;
    }
    rc = fft3d_c2r(pl, pl->h_cplx, pl->h_real, pl->h_work, st);
    if (rc != FFT3D_OK) return rc;
    if (cudaMemcpyAsync(h_out, pl->h_real, fft3d_real_bytes(pl), cudaMemcpyDeviceToHost, st) != cudaSuccess ||
        cudaStreamSynchronize(st) != cudaSuccess) {
        cudaGetLastError();
        return FFT3D_ECUDA;
    }
    return FFT3D_OK;
}

int fft3d_c2c_host(fft3d_plan_t* pl, const void* h_in, void* h_out, int direction) {
    if (pl == nullptr || pl->kind != 1 || h_in == nullptr || h_out == nullptr) return FFT3D_EINVAL;
    if (wrong_device(pl)) return FFT3D_EINVAL;          // the current device is not the plan's
    if (direction != -1 && direction != 1) return FFT3D_EINVAL;
    int rc = ensure_host_buffers(pl);
    if (rc != FFT3D_OK) return rc;
    cudaStream_t st = pl->h_stream;
    const size_t cb = fft3d_complex_bytes(pl);
    if (cudaMemcpyAsync(pl->h_real, h_in, cb, cudaMemcpyHostToDevice, st) != cudaSuccess) {
        cudaGetLastError();
        return FFT3D_ECUDA;
    }
    rc = fft3d_c2c(pl, pl->h_real, pl->h_cplx, pl->h_work, direction, st);
    if (rc != FFT3D_OK) return rc;
    if (cudaMemcpyAsync(h_out, pl->h_cplx, cb, cudaMemcpyDeviceToHost, st) != cudaSuccess ||
        cudaStreamSynchronize(st) != cudaSuccess) {
        cudaGetLastError();
        return FFT3D_ECUDA;
    }
    return FFT3D_OK;
}

int fft3d_destroy(fft3d_plan_t* pl) {
    if (pl == nullptr) return FFT3D_OK;
    cudaFree(pl->tw_zb); cudaFree(pl->tw_zc); cudaFree(pl->tw_y2); cudaFree(pl->tw_x2); cudaFree(pl->tw_x4); cudaFree(pl->tw_z); cudaFree(pl->tw_y); cudaFree(pl->tw_x); cudaFree(pl->twz);
    cudaFree(pl->h_real); cudaFree(pl->h_cplx); cudaFree(pl->h_work);
    if (pl->h_stream) cudaStreamDestroy(pl->h_stream);
    timing_free(pl);
    cudaGetLastError();
    delete pl;
    return FFT3D_OK;
}

const char* fft3d_strerror(int status) {
    switch (status) {
        case FFT3D_OK: return "ok";
        case FFT3D_EINVAL: return "invalid argument (extents, virtual_slabs, dtype, pointers or aliasing)";
        case FFT3D_EUNSUPPORTED: return "unsupported extent (need Nz even; Nx, Ny, Nz/2 of the form 2^a, 3*2^a, 5*2^a or 7*2^a within the built range)";
        case FFT3D_ENOMEM: return "out of memory";
        case FFT3D_ECUDA: return "CUDA error (no device, or a launch/runtime failure)";
        case FFT3D_EWORKSPACE: return "workspace too small or misaligned";
        default: return "unknown status";
    }
}

}  // extern "C"
