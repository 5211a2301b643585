// fft3d_static.cu -- fft3d_r2c_static: the forward R2C transform for callers that cannot allocate device memory.
//
// Who this is for.  Every other compute call of this library needs two things the caller must get from the CUDA
// allocator: a plan (fft3d_plan uploads its twiddle tables into cudaMalloc'ed buffers) and an array-sized
// workspace.  Some callers have no allocator to ask:
//   * a plug-in running inside a host application whose memory pool took the whole card at start-up, so that a raw
//     cudaMalloc simply fails (or is forbidden by the host's rules);
//   * a steady-state loop (in-situ analysis inside a solver's time step, a serving loop) where cudaMalloc and
//     cudaFree are ruled out because they synchronise the whole device and can fail when the card is full;
//   * a process confined to a fixed memory budget that was handed its input and output buffers and nothing else.
// For them this file carries its own scratch: one file-scope array in device memory, part of the library image, of
// FFT3D_STATIC_SCRATCH_BYTES (17 MiB).  The caller passes only the input and the output; the call takes no plan,
// creates none, and calls no cudaMalloc / cudaFree / other allocating routine.  The price is a size limit
// (the intermediate array plus the twiddle tables must fit the 17 MiB) and the plain-load kernels (no TMA
// pipelines, no fused z+y pass): this is a path for small grids, not the fast path.
//
// What it computes: exactly fft3d_r2c (Eq. (1); steps 1-5) -- z-axis R2C into the
// output buffer (used as scratch), y-axis C2C with the slab permutation into the intermediate array, x-axis C2C
// into the output, then the split of the packed column 0 into the planes kz = 0 and kz = Nz/2.  The kernels are
// the library's plain-load ones (what fft3d_set_variant(plan, 1) selects) and the twiddle tables are built by the
// same formulas, so the result equals that variant's.
//
// The scratch array and its address.  `g_static_scratch` below is a `__device__` variable.  Inside host code that
// NAME is only the host-side handle the runtime registers for the symbol -- it is not a device address, and a kernel
// handed `g_static_scratch` (or `&g_static_scratch[0]`) from host code would fault, or scribble over host memory
// on a system where the GPU can reach it.  The device address is a per-device fact (every device that loads this
// module gets its own copy of the array), so it is asked for once per device, with that device current, through
// cudaGetSymbolAddress, and cached in `g_dev[device]`.  That query (and the module load it can trigger) happens in
// the FIRST call on a device: make that call during start-up, outside any stream capture.
//
// Sharing.  There is one array per device and every call on that device uses it: two calls whose GPU work can
// overlap (different streams, or different host threads on different streams) race on it and corrupt each other.
// Calls on one stream are safe, whatever their shapes: a change of shape re-uploads the tables and every call
// rewrites the intermediate array, all in stream order.  The array keeps whatever the previous call left.  That is
// relied on for the tables (a run of calls with one shape uploads them once) and harmless for the rest: no part of
// the array has to start at zero, because the intermediate array is written in full by the y pass before the x pass
// reads it -- so nothing is cleared.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdint>
#include <cstring>
#include <mutex>
#include <vector>

#include "../../include/fft3d.h"
#include "fft_kernels.cuh"
#include "fft_registry.h"

namespace fft3d {
// plane-sized fix-up kernel of fft3d_fixup.cu (same declaration as in fft3d_plan.cu)
struct PlaneArgs {
    const void* src;
    void* dst;
    int Nx, Ny, L, M;
};
cudaError_t launch_unpack_nyquist(int dtype, const PlaneArgs& a, cudaStream_t st);
}  // namespace fft3d

using namespace fft3d;

// The scratch itself: [ tables (tw_z | tw_y | tw_x | twz, each 256-byte aligned) | intermediate array ].
// Zero-initialised by the loader; 256-byte alignment covers every vector access of the kernels (16 bytes needed).
static __device__ __align__(256) unsigned char g_static_scratch[FFT3D_STATIC_SCRATCH_BYTES];

namespace {

constexpr int kMaxDevices = 64;
constexpr size_t kAlign = 256;

struct DeviceState {
    unsigned char* base;                  // DEVICE address of g_static_scratch on this device (nullptr: not asked yet)
    int num_sms;
    // what the cached host tables and grid sizes below were built for
    long long Nx, Ny, Nz;
    int dtype;
    std::vector<unsigned char> tables;    // host image of the table region
    size_t off_z, off_y, off_x, off_twz;  // byte offsets inside it
    int grid_z, grid_y, grid_x;
    bool resident;                        // the device copy of the table region holds these tables
};

std::mutex g_mu;                          // host-side: one enqueue at a time (the GPU-side race is the caller's to avoid)
DeviceState g_dev[kMaxDevices];

size_t align_up(size_t v) { return (v + kAlign - 1) & ~(kAlign - 1); }

const long double kTwoPi = 6.283185307179586476925286766559005768L;

// exp(-2 pi i num/den) with the fraction reduced first and the axis values exact
void unit_root(long long num, long long den, long double* c, long double* s) {
    const long long m = ((num % den) + den) % den;
    const long double a = kTwoPi * (long double)m / (long double)den;
    *c = cosl(a);
    *s = -sinl(a);
    if (m == 0) { *c = 1; *s = 0; }
    else if (2 * m == den) { *c = -1; *s = 0; }
    else if (4 * m == den) { *c = 0; *s = -1; }
    else if (4 * m == 3 * den) { *c = 0; *s = 1; }
}

void put(unsigned char* dst, size_t i, int esize, long double c, long double s) {
    if (esize == 4) { float* p = reinterpret_cast<float*>(dst) + 2 * i; p[0] = (float)c; p[1] = (float)s; }
    else { double* p = reinterpret_cast<double*>(dst) + 2 * i; p[0] = (double)c; p[1] = (double)s; }
}

size_t stage_table_bytes(const KernelSet* k, int esize) { return (size_t)(k->twn > 0 ? k->twn : 1) * 2 * esize; }

// Stage tables of fft_core.cuh: stage s >= 1, entry (i-1)*Ns + k = exp(-2 pi i * i*k/(Ns*r)), stages back to back.
void fill_stage_table(unsigned char* dst, const KernelSet* k, int esize) {
    size_t off = 0;
    long long Ns = k->radix[0];
    for (int s = 1; s < k->nst; ++s) {
        const int r = k->radix[s];
        for (int i = 1; i < r; ++i)
            for (long long kk = 0; kk < Ns; ++kk) {
                long double c, sn;
                unit_root((long long)i * kk, Ns * r, &c, &sn);
                put(dst, off + (size_t)(i - 1) * Ns + kk, esize, c, sn);
            }
        off += (size_t)(r - 1) * Ns;
        Ns *= r;
    }
}

// dynamic shared memory opt-in (a per-device attribute of the function) and the persistent grid size
int prepare(const void* fn, int threads, size_t smem, int num_sms, int* grid) {
    if (fn == nullptr) return FFT3D_EUNSUPPORTED;
    int occ = 0;
    if (cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess ||
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, fn, threads, smem) != cudaSuccess || occ < 1) {
        cudaGetLastError();
        return FFT3D_ECUDA;
    }
    *grid = occ * num_sms;
    return FFT3D_OK;
}

template <class Args>
int enqueue(const void* fn, long long work_items, int grid_cap, int threads, size_t smem, Args* args, cudaStream_t st) {
    if (work_items <= 0) return FFT3D_OK;
    const long long g = work_items < grid_cap ? work_items : grid_cap;
    void* argv[1] = {args};
    if (cudaLaunchKernel(fn, dim3((unsigned)g), dim3((unsigned)threads), argv, smem, st) != cudaSuccess) {
        cudaGetLastError();
        return FFT3D_ECUDA;
    }
    return FFT3D_OK;
}

bool ranges_overlap(const void* a, size_t na, const void* b, size_t nb) {
    const uintptr_t x = (uintptr_t)a, y = (uintptr_t)b;
    return x < y + nb && y < x + na;
}

}  // namespace

extern "C" int fft3d_r2c_static(long long Nx, long long Ny, long long Nz, int dtype, int virtual_slabs,
                                const void* d_real_in, void* d_cplx_out, void* cuda_stream) {
    // ---- arguments: the same rules as fft3d_plan + fft3d_r2c ----
    if (dtype != FFT3D_F32 && dtype != FFT3D_F64) return FFT3D_EINVAL;
    if (Nx < 2 || Ny < 2 || Nz < 2 || virtual_slabs < 1) return FFT3D_EINVAL;
    if (Nx % virtual_slabs != 0 || Ny % virtual_slabs != 0) return FFT3D_EINVAL;
    if (d_real_in == nullptr || d_cplx_out == nullptr) return FFT3D_EINVAL;
    if (((uintptr_t)d_real_in | (uintptr_t)d_cplx_out) & 15) return FFT3D_EINVAL;
    if (Nz % 2 != 0) return FFT3D_EUNSUPPORTED;
    const long long M = Nz / 2, L = Ny / virtual_slabs;
    const int esize = dtype == FFT3D_F32 ? 4 : 8;
    const KernelSet* kz = find_kernels(M, dtype);
    const KernelSet* ky = find_kernels(Ny, dtype);
    const KernelSet* kx = find_kernels(Nx, dtype);
    if (kz == nullptr || ky == nullptr || kx == nullptr) return FFT3D_EUNSUPPORTED;
    const void* fn_z = kz->z_fn[0];
    const void* fn_y = ky->s_fn[0][KIND_LIN_SLAB];
    const void* fn_x = kx->s_fn[0][KIND_LIN_LIN];
    if (fn_z == nullptr || fn_y == nullptr || fn_x == nullptr) return FFT3D_EUNSUPPORTED;

    // ---- does it fit the built-in scratch?  (checked before anything touches the device) ----
    const size_t off_z = 0;
    const size_t off_y = off_z + align_up(stage_table_bytes(kz, esize));
    const size_t off_x = off_y + align_up(stage_table_bytes(ky, esize));
    const size_t off_twz = off_x + align_up(stage_table_bytes(kx, esize));
    const size_t tables_bytes = off_twz + align_up((size_t)M * 2 * esize);
    // Nx*Ny*M*2*esize, refusing anything that cannot fit before the product can overflow
    const long double want = (long double)Nx * (long double)Ny * (long double)M * 2.0L * esize;
    if (want + (long double)tables_bytes > (long double)FFT3D_STATIC_SCRATCH_BYTES) return FFT3D_EWORKSPACE;
    const size_t rb = (size_t)Nx * Ny * Nz * esize, cb = (size_t)Nx * Ny * (M + 1) * 2 * esize;
    if (ranges_overlap(d_real_in, rb, d_cplx_out, cb)) return FFT3D_EINVAL;

    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return FFT3D_ECUDA; }
    if (dev < 0 || dev >= kMaxDevices) return FFT3D_EUNSUPPORTED;
    cudaStream_t st = (cudaStream_t)cuda_stream;

    std::lock_guard<std::mutex> lock(g_mu);
    DeviceState& ds = g_dev[dev];

    // ---- once per device: where does THIS device keep the array? ----
    if (ds.base == nullptr) {
        void* p = nullptr;
        // not `p = g_static_scratch`: in host code that name is the registration handle, not device memory
        if (cudaGetSymbolAddress(&p, g_static_scratch) != cudaSuccess || p == nullptr) {
            cudaGetLastError();
            return FFT3D_ECUDA;
        }
        int sms = 0;
        if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms < 1) {
            cudaGetLastError();
            return FFT3D_ECUDA;
        }
        ds.num_sms = sms;
        ds.dtype = -1;
        ds.base = static_cast<unsigned char*>(p);
    }
    if (ranges_overlap(d_real_in, rb, ds.base, FFT3D_STATIC_SCRATCH_BYTES) ||
        ranges_overlap(d_cplx_out, cb, ds.base, FFT3D_STATIC_SCRATCH_BYTES)) return FFT3D_EINVAL;

    // ---- per shape (host memory only): twiddle tables and grid sizes, kept until the shape changes ----
    if (ds.dtype != dtype || ds.Nx != Nx || ds.Ny != Ny || ds.Nz != Nz) {
        ds.dtype = -1;                                   // invalid until everything below has succeeded
        ds.resident = false;
        int rc = prepare(fn_z, kz->z_threads, kz->z_smem, ds.num_sms, &ds.grid_z);
        if (rc == FFT3D_OK) rc = prepare(fn_y, ky->s_threads, ky->s_smem, ds.num_sms, &ds.grid_y);
        if (rc == FFT3D_OK) rc = prepare(fn_x, kx->s_threads, kx->s_smem, ds.num_sms, &ds.grid_x);
        if (rc != FFT3D_OK) return rc;
        try {
            ds.tables.assign(tables_bytes, 0);
        } catch (...) {
            return FFT3D_ENOMEM;                         // host memory
        }
        unsigned char* t = ds.tables.data();
        fill_stage_table(t + off_z, kz, esize);
        fill_stage_table(t + off_y, ky, esize);
        fill_stage_table(t + off_x, kx, esize);
        for (long long k = 0; k < M; ++k) {              // exp(-2 pi i k / Nz), k < M: the Hermitian step of the z pass
            long double c, s;
            unit_root(k, Nz, &c, &s);
            put(t + off_twz, (size_t)k, esize, c, s);
        }
        ds.off_z = off_z; ds.off_y = off_y; ds.off_x = off_x; ds.off_twz = off_twz;
        ds.Nx = Nx; ds.Ny = Ny; ds.Nz = Nz; ds.dtype = dtype;
    }

    // ---- the call proper, all on the caller's stream ----
    // Tables first, whenever the device copy is not this shape's (first call, or the previous call on this device was
    // for another shape); a loop over one shape uploads once and then finds them where the last call left them.  The
    // copy is ordered on the caller's stream like the kernels; its source is pageable host memory, which the runtime
    // has staged by the time cudaMemcpyAsync returns (it may first wait for earlier work on that stream).
    unsigned char* d_tables = ds.base;
    unsigned char* d_slab = ds.base + tables_bytes;      // tables_bytes is a multiple of 256
    if (!ds.resident) {
        if (cudaMemcpyAsync(d_tables, ds.tables.data(), tables_bytes, cudaMemcpyHostToDevice, st) != cudaSuccess) {
            cudaGetLastError();
            return FFT3D_ECUDA;
        }
        ds.resident = true;
    }

    // F1 (step 1, z half): real rows -> packed complex rows [Nx][Ny][M], in the caller's output buffer
    ZArgs z{};
    z.in = d_real_in; z.out = d_cplx_out; z.tw = d_tables + ds.off_z; z.twz = d_tables + ds.off_twz;
    z.nrows = Nx * Ny; z.scale = 1.0; z.in_pitch = z.out_pitch = M;
    int rc = enqueue(fn_z, (z.nrows + kz->z_rpb - 1) / kz->z_rpb, ds.grid_z, kz->z_threads, kz->z_smem, &z, st);
    if (rc != FFT3D_OK) return rc;

    // F2 (step 1, y half + steps 2-4): y-axis FFT, row ky stored at slab[q][x][ky % L][M]
    StridedArgs a{};
    a.in = d_cplx_out; a.out = d_slab; a.col0 = nullptr; a.tw = d_tables + ds.off_y;
    a.ntz = (int)((M + ky->tc - 1) / ky->tc); a.ncols = (int)M; a.a_lo = 1; a.L = (int)L;
    a.ntiles = Nx * a.ntz;
    a.in_hi = Ny * M; a.in_lo = 0; a.in_rq = 0; a.in_rl = M;
    a.out_hi = L * M; a.out_lo = 0; a.out_rq = Nx * L * M; a.out_rl = M;
    rc = enqueue(fn_y, a.ntiles, ds.grid_y, ky->s_threads, ky->s_smem, &a, st);
    if (rc != FFT3D_OK) return rc;

    // F3 (step 5): x-axis FFT inside every virtual slab, slab (pitch M) -> output (pitch M+1)
    StridedArgs b{};
    b.in = d_slab; b.out = d_cplx_out; b.col0 = nullptr; b.tw = d_tables + ds.off_x;
    b.ntz = (int)((M + kx->tc - 1) / kx->tc); b.ncols = (int)M; b.a_lo = (int)L; b.L = (int)Nx;
    b.ntiles = (long long)virtual_slabs * L * b.ntz;
    b.in_hi = Nx * L * M; b.in_lo = M; b.in_rq = 0; b.in_rl = L * M;
    b.out_hi = Nx * L * (M + 1); b.out_lo = M + 1; b.out_rq = 0; b.out_rl = L * (M + 1);
    rc = enqueue(fn_x, b.ntiles, ds.grid_x, kx->s_threads, kx->s_smem, &b, st);
    if (rc != FFT3D_OK) return rc;

    // column 0 holds (plane kz = 0) + i (plane kz = Nz/2): separate them in place (Eq. (3)/(4))
    PlaneArgs f{};
    f.src = nullptr; f.dst = d_cplx_out; f.Nx = (int)Nx; f.Ny = (int)Ny; f.L = (int)L; f.M = (int)M;
    if (launch_unpack_nyquist(dtype, f, st) != cudaSuccess) { cudaGetLastError(); return FFT3D_ECUDA; }
    return FFT3D_OK;
}
