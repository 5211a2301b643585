/*
 * fft3d.h -- C ABI of the B200-native slab-decomposed 3D real-to-complex / complex-to-real FFT.
 *
 * The operation is the one "Scalable Multi-node Fast Fourier Transform on GPUs"
 * (arXiv 2202.12756) distributes over p GPUs; here the p slabs are VIRTUAL and live on one
 * GPU, so the paper's MPI all-to-all becomes a layout permutation that is folded into the
 * FFT passes.  Citations: P:n = PAPER.md line n (the paper's text), D:x = DESIGN.md section.
 *
 *   forward  F(kx,ky,kz) = sum_j f(jx,jy,jz) exp(-2 pi i [jx kx/Nx + jy ky/Ny + jz kz/Nz])
 *            kx in [0,Nx), ky in [0,Ny), kz in [0,Nz/2]         Eq. (1), Eq. (4)
 *            UNNORMALISED.
 *   inverse  f(j) = 1/(Nx Ny Nz) Re sum_{k, full grid} Ft(k) exp(+2 pi i [...]),
 *            Ft = the stored half extended by Ft(kx,ky,kz) = conj F(-kx,-ky,Nz-kz)
 *            for kz > Nz/2                                      Eq. (2), Eq. (3)
 *            NORMALISED by 1/(Nx Ny Nz) (the paper's separately timed "normalization",
 *            P:184; reading R1 in D:3).  Imaginary parts that Eq. (3) makes irrelevant
 *            (the non-Hermitian part of the planes kz=0 and kz=Nz/2) are ignored exactly as
 *            that definition ignores them (reading R8).
 *
 * Pipeline (P:69-77 steps 1-5; inverse = reverse order), each arrow-separated item ONE pass
 * over the array:
 *   forward : z-axis R2C  ->  y-axis C2C + global transpose X (steps 2+3+4)  ->  x-axis C2C
 *   inverse : x-axis C2C  ->  inverse transpose + y-axis C2C  ->  z-axis C2R * 1/(NxNyNz)
 * For large cubic-like fp32 plans the z and y passes of an x-plane run inside one kernel and
 * exchange the plane through an L2-resident ring (two passes per direction; D:5.6).  A 3D
 * complex-to-complex transform over the same layouts is declared further down (D:5.7).
 *
 * LAYOUTS (all dense, row-major, no padding; complex = interleaved (re, im)):
 *   real     f[jx][jy][jz]                    z fastest, x slowest
 *   complex  F[q][kx][ky_l][kz]               q = ky / (Ny/p), ky_l = ky % (Ny/p), kz = 0..Nz/2
 *            i.e. virtual rank q owns [Nx][Ny/p][Nz/2+1] with x stride (Ny/p)(Nz/2+1)
 *            and the p ranks are concatenated.  p = 1 is FFTW's natural order.
 *            fft3d_index() returns the element offset of (kx,ky,kz).
 *
 * OWNERSHIP: the caller owns every data buffer and the stream.  A plan owns only its small
 * device twiddle tables and host metadata.  It belongs to the device that was current when it was
 * created: every compute call returns FFT3D_EINVAL when another device is current.  Transform calls
 * do not change the plan, so one plan may be used from several streams concurrently as long as each
 * call has its own workspace; fft3d_set_variant, fft3d_set_option and fft3d_timing_* DO change it and
 * need exclusive access.  The fused z+y kernels are cooperative launches: if the driver refuses one
 * (SM partitions, MPS limits) the call returns FFT3D_ECUDA; fft3d_set_variant(plan, 2) selects the
 * unfused passes.
 *
 * DEVICE entry points (fft3d_r2c / fft3d_c2r) take DEVICE pointers, 16-byte aligned, and
 * return after enqueueing work on `cuda_stream` (a cudaStream_t passed as void*; NULL = the
 * legacy default stream).  They do not allocate and do not synchronise.  Inputs are
 * preserved.  in == out, or a workspace overlapping either, is rejected (FFT3D_EINVAL).
 *
 * HOST entry points (fft3d_r2c_host / fft3d_c2r_host) take HOST pointers (pinned memory
 * gives the best copy rate, pageable works), allocate device buffers inside the plan on
 * first use (released by fft3d_destroy), copy in, transform, copy out and return when the
 * result is in host memory.
 *
 * ERRORS: every function returns an int status (FFT3D_OK = 0) unless stated; none throws,
 * prints or aborts.  No CPU fallback exists: without a CUDA device every compute call
 * returns FFT3D_ECUDA.
 */
#ifndef FFT3D_H_
#define FFT3D_H_

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct fft3d_plan_s fft3d_plan_t;      /* opaque */

enum { FFT3D_F32 = 0, FFT3D_F64 = 1 };          /* dtype of reals; complex is two of them */

enum {
    FFT3D_OK = 0,
    FFT3D_EINVAL = 1,         /* null pointer, extent < 2, p < 1, p not dividing Nx and Ny,
                                 bad dtype, aliased / misaligned buffers                      */
    FFT3D_EUNSUPPORTED = 2,   /* Nz odd, or an extent this build has no kernel for
                                 (see fft3d_supported_length)                                 */
    FFT3D_ENOMEM = 3,         /* host or device allocation failed                             */
    FFT3D_ECUDA = 4,          /* no device, launch or runtime error (cudaGetLastError cleared) */
    FFT3D_EWORKSPACE = 5      /* fft3d_r2c_static only: the problem needs more scratch than the
                                 library's built-in array holds.  (With a caller-supplied
                                 workspace a short buffer cannot be detected from a bare pointer;
                                 callers size it with fft3d_workspace_bytes.)                 */
};

/* Create a plan for an Nx x Ny x Nz real grid split into `virtual_slabs` = p x-slabs
 * (slab decomposition, p <= Nx).  Requirements (reading R6/R7 in D:3): extents >= 2,
 * Nz even, p >= 1, p | Nx, p | Ny, Nx and Ny in the supported C2C length set and Nz/2 in it
 * too (the z pass runs an Nz/2-point complex FFT on packed even/odd pairs).
 * BASELINE.json: fft3d_plan(Nx,Ny,Nz,dtype,virtual_slabs).  *out is NULL on failure. */
int fft3d_plan(fft3d_plan_t **out, long long Nx, long long Ny, long long Nz,
               int dtype, int virtual_slabs);

/* 1 if this build has a C2C kernel of length n (n = 2^a in 4..4096, 3*2^a in 6..3072, 5*2^a in 20..1280
 * or 7*2^a in 28..1792), else 0. */
int fft3d_supported_length(long long n);

/* Sizes in bytes.  Workspace: the single work buffer shared by R2C and C2R (opt. 1):
 * Nx*Ny*(Nz/2) complex, plus -- for plans whose z and y passes run fused -- a ring of a few
 * yz-planes that lives in L2, one Nx*Ny complex side plane and 2*Nx counters (< 1 % more; the
 * library zeroes the counters itself).  Real: Nx*Ny*Nz reals.  Complex: Nx*Ny*(Nz/2+1) complex. */
size_t fft3d_workspace_bytes(const fft3d_plan_t *plan);
size_t fft3d_real_bytes(const fft3d_plan_t *plan);
size_t fft3d_complex_bytes(const fft3d_plan_t *plan);

/* Element (not byte) offset of F(kx,ky,kz) in the complex array:
 * ((q*Nx + kx)*(Ny/p) + ky % (Ny/p))*(Nz/2+1) + kz, q = ky / (Ny/p); -1 if out of range.
 * This is the composition of the paper's steps 2-4 (derivation in D:2). */
long long fft3d_index(const fft3d_plan_t *plan, long long kx, long long ky, long long kz);

/* Forward R2C, Eq. (1): d_real_in [Nx][Ny][Nz] -> d_cplx_out in the slab layout above.
 * d_work: fft3d_workspace_bytes() bytes.  d_cplx_out may also be used as scratch while the call
 * runs.  2 (fused z+y) or 3 full-array kernel passes + one plane-sized fix-up kernel. */
int fft3d_r2c(const fft3d_plan_t *plan, const void *d_real_in, void *d_cplx_out,
              void *d_work, void *cuda_stream);

/* Inverse C2R, Eq. (2)+(3) scaled by 1/(NxNyNz): d_cplx_in (slab layout) -> d_real_out
 * [Nx][Ny][Nz].  d_real_out may also be used as scratch while the call runs. */
int fft3d_c2r(const fft3d_plan_t *plan, const void *d_cplx_in, void *d_real_out,
              void *d_work, void *cuda_stream);

/* Forward R2C for callers that cannot allocate device memory.
 * Everything above needs the CUDA allocator twice: fft3d_plan cudaMalloc's its twiddle tables, and fft3d_r2c wants an
 * array-sized workspace from the caller.  That shuts out code that has no allocator to turn to -- a plug-in inside an
 * application whose memory pool claimed the whole card at start-up (a raw cudaMalloc fails there, or is against the
 * host's rules), the inner loop of a solver or server where cudaMalloc/cudaFree are banned because they stall the whole
 * device and may fail when the card is full, a process held to a fixed memory budget that owns its input and output
 * buffers and nothing more.  fft3d_r2c_static serves them: no plan, no workspace argument, and not one call to
 * cudaMalloc, cudaFree or any other allocating routine.  Its scratch (the Nx*Ny*(Nz/2) complex intermediate array and
 * four small twiddle tables) is a fixed array of FFT3D_STATIC_SCRATCH_BYTES = 17 MiB compiled into the library image;
 * each GPU on which the library's code gets loaded carries that 17 MiB until the process exits, used or not.
 *   Computes exactly what fft3d_plan(Nx,Ny,Nz,dtype,virtual_slabs) + fft3d_r2c compute (Eq. (1), steps 1-5
 * P:69-77, output in the slab layout above), with the plain-load kernels (the ones fft3d_set_variant(plan, 1) picks):
 * it is meant for small grids, not for speed.  d_real_in [Nx][Ny][Nz] and d_cplx_out (Nx*Ny*(Nz/2+1) complex) are the
 * caller's DEVICE buffers on the current device, 16-byte aligned, not overlapping; d_cplx_out doubles as scratch while
 * the call runs, d_real_in is preserved.  Work is enqueued on cuda_stream (NULL = the legacy default stream); the call
 * does not wait for it (only the first call with a new shape may block a little: it copies the tables from pageable host
 * memory, which the runtime orders behind earlier work on that stream).
 *   LIMIT: Nx*Ny*(Nz/2)*sizeof(complex) plus the tables (a few KiB, at most 256 KiB) must fit the 17 MiB: every grid with
 * Nx*Ny*Nz*sizeof(real) <= 16 MiB does (128^3 in fp64, 160^3 or 128x128x256 in fp32).  Larger problems get
 * FFT3D_EWORKSPACE and nothing is launched.  Other errors as for fft3d_plan / fft3d_r2c (FFT3D_EINVAL,
 * FFT3D_EUNSUPPORTED, FFT3D_ECUDA).
 *   FIRST CALL ON A DEVICE: looks up where that device keeps the array (and may make the driver load the library's
 * device code).  Issue it once per device during start-up, with that device current, before any stream capture begins.
 *   SHARING: one array per device serves every call.  Calls queued on the same stream are fine, whatever their shapes.
 * Calls whose GPU work can overlap -- two streams, or two host threads on two streams -- write the same scratch and
 * corrupt each other: serialise them (one stream, or events).  The array is never cleared between calls and need not
 * be: the intermediate array is written in full before it is read, and the tables are left in place on purpose, so that a
 * run of calls with one shape uploads them once (a change of shape uploads the new ones, in stream order). */
#define FFT3D_STATIC_SCRATCH_BYTES ((size_t)17 << 20)
int fft3d_r2c_static(long long Nx, long long Ny, long long Nz, int dtype, int virtual_slabs,
                     const void *d_real_in, void *d_cplx_out, void *cuda_stream);

/* 3D complex-to-complex transform (in the paper's library R2C, C2C and C2R share one
 * workspace).  fft3d_plan_c2c creates a plan for an Nx x Ny x Nz COMPLEX grid over p virtual
 * x-slabs: same requirements as fft3d_plan except that Nz need not be even: Nx, Ny and Nz must be supported
 * lengths, p | Nx, p | Ny.  Rows of >= 1 KiB in whole tiles run the bulk-pipelined row kernel, all others a
 * plain-load one (fft3d_launch_impl says which).  For such a plan
 * fft3d_complex_bytes = Nx*Ny*Nz complex (input, output), fft3d_workspace_bytes the same,
 * fft3d_real_bytes = 0, fft3d_index(kx,ky,kz) = ((q*Nx + kx)*(Ny/p) + ky % (Ny/p))*Nz + kz.
 * fft3d_c2c: direction -1 = forward, unnormalised, d_in natural [Nx][Ny][Nz] -> d_out in the slab layout
 * [p][Nx][Ny/p][Nz]; direction +1 = inverse scaled by 1/(NxNyNz), slab layout -> natural.  Three full-array
 * passes (z rows, y lines with the slab permutation, x lines), or two where the z and y passes run fused
 * (Nz == Ny; fft3d_set_variant applies as for R2C plans).  d_out is also used as scratch; d_in is
 * preserved; all pointers 16-byte aligned device pointers, no overlap; asynchronous on the stream.
 * fft3d_r2c / fft3d_c2r reject a C2C plan with FFT3D_EINVAL and vice versa. */
int fft3d_plan_c2c(fft3d_plan_t **plan_out, long long Nx, long long Ny, long long Nz,
                   int dtype, int virtual_slabs);
int fft3d_c2c(const fft3d_plan_t *plan, const void *d_cplx_in, void *d_cplx_out,
              void *d_work, int direction, void *cuda_stream);

/* Padded in-place layout (P:67 counts Nx/p x Ny x (Nz/2+1) "data points" per GPU: FFTW's in-place
 * convention).  ONE buffer of fft3d_complex_bytes() holds the real field as rows of Nz+2 reals,
 *     f[jx][jy][jz] at ((jx*Ny + jy)*(Nz+2) + jz), the last two reals of a row unused,
 * and, after fft3d_r2c_inplace, its half spectrum in the slab layout [p][Nx][Ny/p][Nz/2+1] (p = 1: F[kx][ky][kz]
 * over the same rows).  fft3d_c2r_inplace is the inverse (scaled by 1/(NxNyNz)); it overwrites the spectrum.
 * d_work: fft3d_workspace_bytes() bytes (the slab array + one Nx*Ny complex plane).  Same extents as fft3d_plan.
 * Rows of this layout start on 8-byte boundaries in fp32, so its z pass and the natural side of its y pass run the
 * plain-load kernels (fft3d_launch_impl reports "plain"); expect ~1.3x the time of the out-of-place transform.
 * fft3d_r2c / fft3d_c2r reject such a plan and vice versa (FFT3D_EINVAL). */
int fft3d_plan_inplace(fft3d_plan_t **plan_out, long long Nx, long long Ny, long long Nz, int dtype, int virtual_slabs);
int fft3d_r2c_inplace(const fft3d_plan_t *plan, void *d_data, void *d_work, void *cuda_stream);
int fft3d_c2r_inplace(const fft3d_plan_t *plan, void *d_data, void *d_work, void *cuda_stream);

/* Pencil layout (p = px x py ranks, each holding (Nx/px) x (Ny/py) x Nz real points --
 * the paper describes this decomposition and does not build it; reading R17 in D:3 fixes the layout).  A second VIRTUAL
 * layout of the same transform: fft3d_r2c leaves the half spectrum as a px x py rank grid would hold it after the
 * standard two-exchange scheme, rank (a, b) owning
 *     F[kx][ky_l][kz_l],  ky = a*Ny/px + ky_l,  kz = b*Nz/(2 py) + kz_l,      [Nx][Ny/px][cz_b]
 * with cz_b = Nz/(2 py) columns, the last rank column b = py-1 also holding the Nyquist column kz = Nz/2 (cz = Nz/(2 py)+1);
 * x is the slowest index inside a rank (stride (Ny/px)*cz_b) and the ranks are concatenated in the order
 * r = a*py + b.  fft3d_index() returns that offset; py = 1 is the slab layout with virtual_slabs = px.  fft3d_c2r takes
 * the same layout back.  Requirements: those of fft3d_plan with p = px, and py | Ny, py | Nz/2, py <= 64.
 * Implementation: the slab transform with p = px, its rows cut into the py column ranges by one more pass over the
 * spectrum ("pencil_split" / "pencil_merge" in fft3d_launch_name); the slab-layout spectrum is staged in the workspace,
 * so fft3d_workspace_bytes() is larger by fft3d_complex_bytes().  Sizes and all other calls as for fft3d_plan. */
int fft3d_plan_pencil(fft3d_plan_t **plan_out, long long Nx, long long Ny, long long Nz, int dtype, int px, int py);

/* ---- Slab decomposition over G GPUs, one process and one plan per GPU -------------------------
 * This is the paper's method itself (P:54 slabs along x; P:67-77 steps 1-5; P:86 inverse), with its exchange fused
 * into the y pass.  Rank r of G owns
 *     real slab     f[x_l][jy][jz],            x = r*Nx/G + x_l          [Nx/G][Ny][Nz]
 *     spectrum part F[kx][ky_l][kz],           ky = r*Ny/G + ky_l        [Nx][Ny/G][Nz/2+1]    (Fig. 1(f))
 * i.e. part r of the layout [G][Nx][Ny/G][Nz/2+1] that a single-GPU plan with virtual_slabs = G produces; results
 * are bit-identical to that plan's.  The stages, each asynchronous on the caller's stream; "==" marks a point
 * where every rank must have finished the previous stage (a barrier, or the collective itself):
 *   forward  fft3d_dist_fwd_local   steps 1-3: z R2C + y C2C of the own planes; row ky of plane x is stored straight
 *                                   to its place in the exchange array (the local transpose, the all-to-all and the
 *                                   chunk transpose, as addressing of the y pass's stores)
 *            ==  [CHUNKS layout: all-to-all of the G chunks]
 *            fft3d_dist_fwd_x       step 5: x C2C on the own y-slab -> own spectrum part
 *            fft3d_dist_fwd_col0    publish the packed column 0 of the own rows as a dense [Nx][Ny/G] plane part
 *            ==  [all-gather of the plane parts, or peer pointers]
 *            fft3d_dist_fwd_unpack  planes kz = 0 and kz = Nz/2 of the own rows (needs C(-kx,-ky): another rank's)
 *   inverse  fft3d_dist_inv_planes  publish the planes kz = 0, Nz/2 of the own rows, [2][Nx][Ny/G]
 *            ==  [all-gather / peer pointers]
 *            fft3d_dist_inv_pack    Hermitian part of the two planes (reading R8) -> packed column, in d_work
 *            fft3d_dist_inv_x       x C2C inverse on the own y-slab -> own part of the exchange array
 *            ==  [CHUNKS layout: all-to-all]
 *            fft3d_dist_inv_local   y C2C inverse + z C2R with 1/(NxNyNz) of the own planes -> own real slab
 * Exchange array, two layouts:
 *   FFT3D_XCHG_UNIFIED  one array [G][Nx][Ny/G][Nz/2] (packed complex) whose part q lives in rank q's memory: the
 *                       forward y pass PUSHES rows into the peers' parts over NVLink (device to device, the
 *                       self chunk like any other), the inverse y pass PULLS them.  d_xchg is the base of the whole
 *                       array as mapped in this process (fft3d_vmm_* maps the peers' allocations into one virtual
 *                       range; on one GPU it is simply one buffer, which is how the tests emulate G ranks).
 *   FFT3D_XCHG_CHUNKS   a local array [G][Nx/G][Ny/G][Nz/2]: chunk q is the message for rank q; the caller
 *                       runs the all-to-all (NCCL ncclSend/ncclRecv pairs) between the stages; after it the G received
 *                       chunks, in source-rank order, ARE the part [Nx][Ny/G][Nz/2] (forward), and vice versa.
 * fft3d_dist_fwd_x / fft3d_dist_inv_x take the own part [Nx][Ny/G][Nz/2] (UNIFIED: d_xchg + rank*FFT3D_DIST_SLAB bytes).
 * Buffer sizes: fft3d_dist_bytes(plan, FFT3D_DIST_REAL | _SLAB (one part of the exchange array) | _SPEC | _PLANES
 * (a plane part, [2][Nx][Ny/G] complex) | _WORK).  d_plane_parts: HOST array of G device pointers, entry q = rank
 * q's plane part as addressable from this device.  G <= 16; G | Nx and G | Ny; all pointers 16-byte
 * aligned device pointers.  fft3d_r2c / fft3d_c2r reject a distributed plan and vice versa (FFT3D_EINVAL). */
enum { FFT3D_DIST_REAL = 0, FFT3D_DIST_SLAB = 1, FFT3D_DIST_SPEC = 2, FFT3D_DIST_PLANES = 3, FFT3D_DIST_WORK = 4 };
enum { FFT3D_XCHG_UNIFIED = 0, FFT3D_XCHG_CHUNKS = 1 };
int fft3d_plan_dist(fft3d_plan_t **plan_out, long long Nx, long long Ny, long long Nz, int dtype, int G, int rank);
size_t fft3d_dist_bytes(const fft3d_plan_t *plan, int which);
int fft3d_dist_fwd_local(const fft3d_plan_t *plan, const void *d_real_slab, void *d_xchg, int layout, void *d_work,
                         void *cuda_stream);
int fft3d_dist_fwd_x(const fft3d_plan_t *plan, const void *d_slab_part, void *d_spec_part, void *cuda_stream);
int fft3d_dist_fwd_col0(const fft3d_plan_t *plan, const void *d_spec_part, void *d_plane_part, void *cuda_stream);
int fft3d_dist_fwd_unpack(const fft3d_plan_t *plan, void *d_spec_part, const void *const *d_plane_parts, void *cuda_stream);
int fft3d_dist_inv_planes(const fft3d_plan_t *plan, const void *d_spec_part, void *d_plane_part, void *cuda_stream);
int fft3d_dist_inv_pack(const fft3d_plan_t *plan, const void *const *d_plane_parts, void *d_work, void *cuda_stream);
int fft3d_dist_inv_x(const fft3d_plan_t *plan, const void *d_spec_part, void *d_slab_part, void *d_work, void *cuda_stream);
int fft3d_dist_inv_local(const fft3d_plan_t *plan, const void *d_xchg, int layout, void *d_real_slab, void *d_work,
                         void *cuda_stream);

/* One virtual address range over G device allocations (CUDA virtual memory management) for the UNIFIED exchange
 * array: every rank creates its part (`bytes` a multiple of fft3d_vmm_granularity(); *fd_out, if asked for, is a POSIX
 * file descriptor the owner passes to its peers and closes afterwards), imports the peers' descriptors, and maps all
 * G handles back to back in rank order: *va_out + q*part_bytes is then rank q's memory, readable and writable from
 * the current device (NVLink peer access; the same device in the single-GPU tests).  Handles are plain integers
 * (CUmemGenericAllocationHandle).  Unmap before releasing; a part stays alive while any rank holds a handle. */
size_t fft3d_vmm_granularity(void);
int fft3d_vmm_create(size_t bytes, unsigned long long *handle_out, int *fd_out);
int fft3d_vmm_import(int fd, unsigned long long *handle_out);
int fft3d_vmm_map(const unsigned long long *handles, int n, size_t part_bytes, void **va_out);
int fft3d_vmm_unmap(void *va, int n, size_t part_bytes);
int fft3d_vmm_release(unsigned long long handle);

/* Host-buffer variant of fft3d_c2c (as fft3d_r2c_host below): H2D copy, transform, D2H copy, synchronous. */
int fft3d_c2c_host(fft3d_plan_t *plan, const void *h_cplx_in, void *h_cplx_out, int direction);

/* Host-buffer variants: H2D copy, transform, D2H copy, synchronous.  The plan lazily
 * allocates real + complex + workspace device buffers (fft3d_real_bytes + fft3d_complex_bytes
 * + fft3d_workspace_bytes) and keeps them until fft3d_destroy. */
int fft3d_r2c_host(fft3d_plan_t *plan, const void *h_real_in, void *h_cplx_out);
int fft3d_c2r_host(fft3d_plan_t *plan, const void *h_cplx_in, void *h_real_out);

/* Number of kernels one fft3d_r2c (which = 0) or fft3d_c2r (which = 1) call launches, and the
 * name of launch i (a static string; NULL if i is out of range).  Names: "z_r2c", "y_c2c_fwd",
 * "x_c2c_fwd", "nyquist_unpack", "pencil_split", "pencil_merge" (pencil-layout plans), "nyquist_pack", "x_c2c_inv", "x_c2c_inv_col0" (the packed
 * column 0 of the inverse x pass, TMA path only), "y_c2c_inv", "z_c2r", and -- when the z and y
 * passes of a plane run as one kernel through an L2-resident ring --
 * "zy_r2c_fused" (paper step 1 + steps 2-4) and "yz_c2r_fused" (their reverse); C2C plans:
 * "z_c2c_fwd", "y_c2c_fwd", "x_c2c_fwd" (which = 0) and "x_c2c_inv", "y_c2c_inv", "z_c2c_inv" (which = 1), or
 * "zy_c2c_fused_fwd", "x_c2c_fwd" and "x_c2c_inv", "yz_c2c_fused_inv" when fused. */
int fft3d_launches(const fft3d_plan_t *plan, int which);
const char *fft3d_launch_name(const fft3d_plan_t *plan, int which, int i);

/* Which implementation launch i runs with the plan's current variant (a static string; NULL if i is out of
 * range): "fused_ring" (z+y passes of a plane in one persistent kernel, D:5.6), "bulk" (z rows streamed by 1-D
 * bulk copies, D:5.3), "tma" (strided pass on whole tiles through a TMA ring, D:5.2), "tma_split2" /
 * "tma_split4" (the same on half / quarter tiles plus a radix-2 / radix-4 combine), "plain" (plain loads and
 * stores: any extent), "fixup" (the plane-sized Nyquist pack / unpack kernels, D:5.4).  Tests use it to make
 * sure a shape really exercises the kernel it is meant to. */
const char *fft3d_launch_impl(const fft3d_plan_t *plan, int which, int i);

/* Per-kernel timing for roofline reports.  After fft3d_timing_enable(plan, max_calls) every
 * fft3d_r2c / fft3d_c2r call on this plan records CUDA events between its kernel launches on the
 * caller's stream (until max_calls calls per direction have been recorded; later calls run
 * untimed).  fft3d_timing_read waits for the recorded events and returns, for direction
 * `which` (0 = r2c, 1 = c2r), the summed duration in ms of each launch slot over the recorded
 * calls (ms_sum[i], i < fft3d_launches(plan, which), in launch order, named by
 * fft3d_launch_name) and the number of calls, then resets the counters.  max_calls = 0 disables
 * timing.  Not thread-safe while enabled. */
#define FFT3D_MAX_LAUNCHES 8
int fft3d_timing_enable(fft3d_plan_t *plan, int max_calls);
int fft3d_timing_read(fft3d_plan_t *plan, int which, float *ms_sum, int *calls);

/* Kernel selection.  variant 0 (default) = the fastest known path for the extents: z and y
 * passes of each x-plane fused into one persistent kernel where that wins (cubic-like fp32
 * plans of >= 2 GiB, Ny == Nz: four array passes per R2C+C2R pair) and TMA-pipelined passes
 * elsewhere; variant 2 = the first-generation unfused TMA-pipelined passes (six array passes per pair; whole
 * tiles even where only one ring stage fits);
 * variant 3 = the fused z+y passes wherever they are compiled (any cubic-like plan with
 * N >= 128); variant 1 = plain-load kernels everywhere (ablation / cross-check).  Variants 0-2
 * without fusion give bit-identical results; the fused kernels run the same butterflies but are
 * compiled separately, so they may differ in the last bit (FMA contraction) -- all variants meet
 * the same error bound.  Returns FFT3D_EINVAL for an unknown variant; affects later calls on
 * this plan.  The workspace size does not depend on the variant. */
int fft3d_set_variant(fft3d_plan_t *plan, int variant);

/* Tunables of the fused z+y pipeline (D:5.6); the defaults are the measured best on B200.  Like
 * fft3d_set_variant these change the plan: call them while no transform on this plan is being enqueued.
 * Results do not depend on them (bit-identical).  Returns FFT3D_EINVAL for an unknown option or a value out
 * of range.
 *   FUSED_MIXED              1 (default): every CTA runs both roles, one consumer group on z tiles and one on y tiles,
 *                            its load warp dealing the ring slots to the two streams; 0: one role per CTA
 *   FUSED_Z_SMS_FWD / _INV   with one role per CTA: SMs [0, value) run the z tiles, the others the y tiles (even;
 *                            0 = alternate CTA pairs)
 *   FUSED_RING_PLANES        yz-planes in the L2 ring (2 .. the number the workspace was sized for)
 *   FUSED_JITTER             stress testing only: every CTA's load warp pauses a pseudo-random 0..value ns (value <= 10^6)
 *                            before each tile, which scrambles the order in which tiles are drawn and taken; the pipeline
 *                            must neither stall nor change a bit of the result.  0 (default) = off */
enum { FFT3D_OPT_FUSED_Z_SMS_FWD = 1, FFT3D_OPT_FUSED_Z_SMS_INV = 2, FFT3D_OPT_FUSED_RING_PLANES = 3, FFT3D_OPT_FUSED_MIXED = 4,
       FFT3D_OPT_FUSED_JITTER = 5 };
int fft3d_set_option(fft3d_plan_t *plan, int option, long long value);

int fft3d_destroy(fft3d_plan_t *plan);          /* NULL is accepted */

const char *fft3d_strerror(int status);         /* static string, never NULL */

#ifdef __cplusplus
}
#endif
#endif /* FFT3D_H_ */
