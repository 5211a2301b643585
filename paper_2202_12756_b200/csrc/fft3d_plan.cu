// fft3d_plan.cu -- the C ABI of include/fft3d.h: plan creation, twiddle tables, and the launch
// sequences of the forward (F1, F2, F3, fix-up) and inverse (pre-pack, I1, I2, I3) transforms.
//
// Pipeline and citations (P:n = PAPER.md line n):
//   F1  z-axis R2C on every row                        step 1, z half
//   F2  y-axis C2C, rows written to the slab layout    step 1, y half + steps 2,3,4
//   F3  x-axis C2C with stride (Ny/p)(Nz/2+1)          step 5
//   inverse: the same in reverse order with 1/(NxNyNz) fused into the last pass.
// One workspace serves both directions (optimisation 1).
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
cudaError_t launch_pack_nyquist(int dtype, const PlaneArgs& a, cudaStream_t st);

}  // namespace fft3d

using namespace fft3d;

struct TimingState {
    int max_calls;
    int calls[2];
    std::vector<cudaEvent_t> ev[2];      // (FFT3D_MAX_LAUNCHES + 1) events per recorded call
};

struct fft3d_plan_s {
    long long Nx, Ny, Nz, M, L;
    int p, dtype, esize;       // esize = bytes per real
    int variant;
    const KernelSet *kz, *ky, *kx;
    void *tw_z, *tw_y, *tw_x, *twz;     // device tables
    int num_sms;
    int grid_z[2], grid_y[2], grid_x[2];   // persistent grid sizes [fwd, inv]
    // buffers of the host-pointer entry points (lazy)
    void *h_real, *h_cplx, *h_work;
    cudaStream_t h_stream;
    TimingState* timing;       // null unless fft3d_timing_enable was called
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
int upload_stage_twiddles(const KernelSet* k, int esize, void** dptr) {
    *dptr = nullptr;
    size_t n = (size_t)(k->twn > 0 ? k->twn : 1);
    std::vector<unsigned char> buf(n * 2 * esize, 0);
    size_t off = 0;
    long long Ns = k->radix[0];
    for (int s = 1; s < k->nst; ++s) {
        int r = k->radix[s];
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

}  // namespace

extern "C" {

int fft3d_supported_length(long long n) {
    return find_kernels(n, FFT3D_F32) != nullptr ? 1 : 0;
}

int fft3d_plan(fft3d_plan_t** out, long long Nx, long long Ny, long long Nz, int dtype, int virtual_slabs) {
    if (out == nullptr) return FFT3D_EINVAL;
    *out = nullptr;
    if (dtype != FFT3D_F32 && dtype != FFT3D_F64) return FFT3D_EINVAL;
    if (Nx < 2 || Ny < 2 || Nz < 2 || virtual_slabs < 1) return FFT3D_EINVAL;
    if (Nx % virtual_slabs != 0 || Ny % virtual_slabs != 0) return FFT3D_EINVAL;
    if (Nz % 2 != 0) return FFT3D_EUNSUPPORTED;
    const KernelSet* kz = find_kernels(Nz / 2, dtype);
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
    pl->Nx = Nx; pl->Ny = Ny; pl->Nz = Nz; pl->M = Nz / 2; pl->p = virtual_slabs; pl->L = Ny / virtual_slabs;
    pl->dtype = dtype; pl->esize = dtype == FFT3D_F32 ? 4 : 8;
    pl->kz = kz; pl->ky = ky; pl->kx = kx; pl->num_sms = sms;

    int rc = upload_stage_twiddles(kz, pl->esize, &pl->tw_z);
    if (rc == FFT3D_OK) rc = upload_stage_twiddles(ky, pl->esize, &pl->tw_y);
    if (rc == FFT3D_OK) rc = upload_stage_twiddles(kx, pl->esize, &pl->tw_x);
    if (rc == FFT3D_OK) rc = upload_z_twiddles(Nz, pl->M, pl->esize, &pl->twz);
    for (int d = 0; d < 2 && rc == FFT3D_OK; ++d) {
        rc = prepare_kernel(kz->z_fn[d], kz->z_threads, kz->z_smem, sms, &pl->grid_z[d]);
        const int ykind = d == 0 ? KIND_LIN_SLAB : KIND_SLAB_LIN;
        if (rc == FFT3D_OK) rc = prepare_kernel(ky->s_fn[d][ykind], ky->s_threads, ky->s_smem, sms, &pl->grid_y[d]);
        if (rc == FFT3D_OK) rc = prepare_kernel(kx->s_fn[d][KIND_LIN_LIN], kx->s_threads, kx->s_smem, sms, &pl->grid_x[d]);
    }
    if (rc != FFT3D_OK) { fft3d_destroy(pl); return rc; }
    *out = pl;
    return FFT3D_OK;
}

size_t fft3d_workspace_bytes(const fft3d_plan_t* pl) {
    return pl ? (size_t)pl->Nx * pl->Ny * pl->M * 2 * pl->esize : 0;
}
size_t fft3d_real_bytes(const fft3d_plan_t* pl) {
    return pl ? (size_t)pl->Nx * pl->Ny * pl->Nz * pl->esize : 0;
}
size_t fft3d_complex_bytes(const fft3d_plan_t* pl) {
    return pl ? (size_t)pl->Nx * pl->Ny * (pl->M + 1) * 2 * pl->esize : 0;
}

long long fft3d_index(const fft3d_plan_t* pl, long long kx, long long ky, long long kz) {
    if (pl == nullptr || kx < 0 || kx >= pl->Nx || ky < 0 || ky >= pl->Ny || kz < 0 || kz > pl->M) return -1;
    const long long q = ky / pl->L, l = ky % pl->L;
    return ((q * pl->Nx + kx) * pl->L + l) * (pl->M + 1) + kz;
}

int fft3d_launches(const fft3d_plan_t* pl, int which) {
    (void)which;
    return pl ? 4 : 0;
}

int fft3d_set_variant(fft3d_plan_t* pl, int variant) {
    if (pl == nullptr || variant != 0) return FFT3D_EINVAL;
    pl->variant = variant;
    return FFT3D_OK;
}

int fft3d_r2c(const fft3d_plan_t* pl, const void* d_in, void* d_out, void* d_work, void* stream) {
    if (pl == nullptr || d_in == nullptr || d_out == nullptr || d_work == nullptr) return FFT3D_EINVAL;
    const size_t rb = fft3d_real_bytes(pl), cb = fft3d_complex_bytes(pl), wb = fft3d_workspace_bytes(pl);
    if (((uintptr_t)d_in | (uintptr_t)d_out | (uintptr_t)d_work) & 15) return FFT3D_EINVAL;
    if (overlap(d_in, rb, d_out, cb) || overlap(d_in, rb, d_work, wb) || overlap(d_out, cb, d_work, wb))
        return FFT3D_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    const long long Nx = pl->Nx, Ny = pl->Ny, M = pl->M, L = pl->L, p = pl->p;

    Recorder rec(pl, 0, st);
    rec.mark(0);
    // F1: real [Nx*Ny rows][Nz] -> packed complex [Nx][Ny][M] in d_out (scratch use)
    ZArgs z{};
    z.in = d_in; z.out = d_out; z.tw = pl->tw_z; z.twz = pl->twz; z.nrows = Nx * Ny; z.scale = 1.0;
    const KernelSet* kz = pl->kz;
    int rc = launch(kz->z_fn[0], (z.nrows + kz->z_rpb - 1) / kz->z_rpb, pl->grid_z[0], kz->z_threads,
                    kz->z_smem, &z, st);
    if (rc != FFT3D_OK) return rc;
    rec.mark(1);

    // F2: y-axis FFT of d_out [x][y][M]; row ky goes to work[q][x][ky_l][M]  (steps 2-4 folded in)
    const KernelSet* ky = pl->ky;
    StridedArgs a{};
    a.in = d_out; a.out = d_work; a.col0 = nullptr; a.tw = pl->tw_y;
    a.ntz = (int)((M + ky->tc - 1) / ky->tc); a.ncols = (int)M; a.a_lo = 1; a.L = (int)L;
    a.ntiles = Nx * a.ntz;
    a.in_hi = Ny * M; a.in_lo = 0; a.in_rq = 0; a.in_rl = M;
    a.out_hi = L * M; a.out_lo = 0; a.out_rq = Nx * L * M; a.out_rl = M;
    rc = launch(ky->s_fn[0][KIND_LIN_SLAB], a.ntiles, pl->grid_y[0], ky->s_threads, ky->s_smem, &a, st);
    if (rc != FFT3D_OK) return rc;
    rec.mark(2);

    // F3: x-axis FFT per virtual slab q and row ky_l: work (pitch M) -> d_out (pitch M+1)
    const KernelSet* kx = pl->kx;
    StridedArgs b{};
    b.in = d_work; b.out = d_out; b.col0 = nullptr; b.tw = pl->tw_x;
    b.ntz = (int)((M + kx->tc - 1) / kx->tc); b.ncols = (int)M; b.a_lo = (int)L; b.L = (int)Nx;
    b.ntiles = (long long)p * L * b.ntz;
    b.in_hi = Nx * L * M; b.in_lo = M; b.in_rq = 0; b.in_rl = L * M;
    b.out_hi = Nx * L * (M + 1); b.out_lo = M + 1; b.out_rq = 0; b.out_rl = L * (M + 1);
    rc = launch(kx->s_fn[0][KIND_LIN_LIN], b.ntiles, pl->grid_x[0], kx->s_threads, kx->s_smem, &b, st);
    if (rc != FFT3D_OK) return rc;
    rec.mark(3);

    // column 0 holds A + iB (planes kz = 0 and kz = Nz/2): separate them in place
    PlaneArgs f{};
    f.src = nullptr; f.dst = d_out; f.Nx = (int)Nx; f.Ny = (int)Ny; f.L = (int)L; f.M = (int)M;
    if (launch_unpack_nyquist(pl->dtype, f, st) != cudaSuccess) { cudaGetLastError(); return FFT3D_ECUDA; }
    rec.mark(4);
    return FFT3D_OK;
}

int fft3d_c2r(const fft3d_plan_t* pl, const void* d_in, void* d_out, void* d_work, void* stream) {
    if (pl == nullptr || d_in == nullptr || d_out == nullptr || d_work == nullptr) return FFT3D_EINVAL;
    const size_t rb = fft3d_real_bytes(pl), cb = fft3d_complex_bytes(pl), wb = fft3d_workspace_bytes(pl);
    if (((uintptr_t)d_in | (uintptr_t)d_out | (uintptr_t)d_work) & 15) return FFT3D_EINVAL;
    if (overlap(d_in, cb, d_out, rb) || overlap(d_in, cb, d_work, wb) || overlap(d_out, rb, d_work, wb))
        return FFT3D_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    const long long Nx = pl->Nx, Ny = pl->Ny, Nz = pl->Nz, M = pl->M, L = pl->L, p = pl->p;

    // pre-pack: side[q][kx][ky_l] = sym(plane kz=0) + i sym(plane kz=Nz/2), kept at the start of
    // the workspace until I1 has consumed it (reading R8: only the Hermitian part of the two
    // self-conjugate planes enters Eq. (2)+(3)).
    Recorder rec(pl, 1, st);
    rec.mark(0);
    PlaneArgs f{};
    f.src = d_in; f.dst = d_work; f.Nx = (int)Nx; f.Ny = (int)Ny; f.L = (int)L; f.M = (int)M;
    if (launch_pack_nyquist(pl->dtype, f, st) != cudaSuccess) { cudaGetLastError(); return FFT3D_ECUDA; }
    rec.mark(1);

    // I1: x-axis inverse FFT: d_in (pitch M+1, column 0 from the side buffer) -> d_out scratch (pitch M)
    const KernelSet* kx = pl->kx;
    StridedArgs b{};
    b.in = d_in; b.out = d_out; b.col0 = d_work; b.tw = pl->tw_x;
    b.ntz = (int)((M + kx->tc - 1) / kx->tc); b.ncols = (int)M; b.a_lo = (int)L; b.L = (int)Nx;
    b.ntiles = (long long)p * L * b.ntz;
    b.in_hi = Nx * L * (M + 1); b.in_lo = M + 1; b.in_rq = 0; b.in_rl = L * (M + 1);
    b.c0_hi = Nx * L; b.c0_lo = 1; b.c0_rl = L;
    b.out_hi = Nx * L * M; b.out_lo = M; b.out_rq = 0; b.out_rl = L * M;
    int rc = launch(kx->s_fn[1][KIND_LIN_LIN], b.ntiles, pl->grid_x[1], kx->s_threads, kx->s_smem, &b, st);
    if (rc != FFT3D_OK) return rc;
    rec.mark(2);

    // I2: y-axis inverse FFT gathering rows from the slab layout: d_out scratch -> work [x][y][M]
    const KernelSet* ky = pl->ky;
    StridedArgs a{};
    a.in = d_out; a.out = d_work; a.col0 = nullptr; a.tw = pl->tw_y;
    a.ntz = (int)((M + ky->tc - 1) / ky->tc); a.ncols = (int)M; a.a_lo = 1; a.L = (int)L;
    a.ntiles = Nx * a.ntz;
    a.in_hi = L * M; a.in_lo = 0; a.in_rq = Nx * L * M; a.in_rl = M;
    a.out_hi = Ny * M; a.out_lo = 0; a.out_rq = 0; a.out_rl = M;
    rc = launch(ky->s_fn[1][KIND_SLAB_LIN], a.ntiles, pl->grid_y[1], ky->s_threads, ky->s_smem, &a, st);
    if (rc != FFT3D_OK) return rc;
    rec.mark(3);

    // I3: z-axis C2R with the 1/(NxNyNz) normalisation: work -> d_out
    const KernelSet* kz = pl->kz;
    ZArgs z{};
    z.in = d_work; z.out = d_out; z.tw = pl->tw_z; z.twz = pl->twz; z.nrows = Nx * Ny;
    z.scale = 1.0 / ((double)Nx * (double)Ny * (double)Nz);
    rc = launch(kz->z_fn[1], (z.nrows + kz->z_rpb - 1) / kz->z_rpb, pl->grid_z[1], kz->z_threads,
                kz->z_smem, &z, st);
    rec.mark(4);
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
    if (pl == nullptr || max_calls < 0 || max_calls > 4096) return FFT3D_EINVAL;
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
    if (cudaStreamCreateWithFlags(&pl->h_stream, cudaStreamNonBlocking) != cudaSuccess) {
        cudaGetLastError();
        return FFT3D_ECUDA;
    }
    if (cudaMalloc(&pl->h_real, fft3d_real_bytes(pl)) != cudaSuccess ||
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
    if (pl == nullptr || h_in == nullptr || h_out == nullptr) return FFT3D_EINVAL;
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
    if (pl == nullptr || h_in == nullptr || h_out == nullptr) return FFT3D_EINVAL;
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

int fft3d_destroy(fft3d_plan_t* pl) {
    if (pl == nullptr) return FFT3D_OK;
    cudaFree(pl->tw_z); cudaFree(pl->tw_y); cudaFree(pl->tw_x); cudaFree(pl->twz);
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
        case FFT3D_EUNSUPPORTED: return "unsupported extent (need Nz even; Nx, Ny, Nz/2 of the form 2^a or 3*2^a within the built range)";
        case FFT3D_ENOMEM: return "out of memory";
        case FFT3D_ECUDA: return "CUDA error (no device, or a launch/runtime failure)";
        case FFT3D_EWORKSPACE: return "workspace too small or misaligned";
        default: return "unknown status";
    }
}

}  // extern "C"
