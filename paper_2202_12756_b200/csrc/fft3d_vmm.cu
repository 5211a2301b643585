// fft3d_vmm.cu -- one virtual address range over allocations that live on different GPUs (CUDA virtual memory
// management), for the UNIFIED exchange array of distributed plans (include/fft3d.h).
//
// The paper exchanges chunks with MPI_Isend/Irecv between device buffers and copies the self
// chunk with cudaMemcpy.  On an NVLink/NVSwitch node every GPU can address every peer's memory, so here
// the exchange array [G][Nx][Ny/G][Nz/2] is ONE array in every rank's address space whose part q is physically
// rank q's memory: each rank creates its part (fft3d_vmm_create, exportable as a POSIX file descriptor), the
// ranks pass the descriptors to one another (SCM_RIGHTS over a Unix socket: paper_2202_12756_b200/dist.py),
// import them (fft3d_vmm_import) and map all G parts back to back (fft3d_vmm_map).  The y pass's tensor-map
// stores then land in the owner's HBM directly -- no pack kernel, no staging copy, no separate all-to-all.
// The driver entry points are resolved at run time (no libcuda link dependency, as for the tensor-map encoder).
#include <cuda.h>
#include <cuda_runtime.h>

#include <cstdint>
#include <new>

#include "../../include/fft3d.h"

namespace {

template <typename F>
bool resolve(const char* name, F* fn) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint(name, &p, cudaEnableDefault, &q) != cudaSuccess || q != cudaDriverEntryPointSuccess || p == nullptr) {
        cudaGetLastError();
        return false;
    }
    *fn = reinterpret_cast<F>(p);
    return true;
}

struct Api {
    CUresult (*create)(CUmemGenericAllocationHandle*, size_t, const CUmemAllocationProp*, unsigned long long);
    CUresult (*release)(CUmemGenericAllocationHandle);
    CUresult (*exportH)(void*, CUmemGenericAllocationHandle, CUmemAllocationHandleType, unsigned long long);
    CUresult (*importH)(CUmemGenericAllocationHandle*, void*, CUmemAllocationHandleType);
    CUresult (*reserve)(CUdeviceptr*, size_t, size_t, CUdeviceptr, unsigned long long);
    CUresult (*addrFree)(CUdeviceptr, size_t);
    CUresult (*map)(CUdeviceptr, size_t, size_t, CUmemGenericAllocationHandle, unsigned long long);
    CUresult (*unmap)(CUdeviceptr, size_t);
    CUresult (*setAccess)(CUdeviceptr, size_t, const CUmemAccessDesc*, size_t);
    CUresult (*granularity)(size_t*, const CUmemAllocationProp*, CUmemAllocationGranularity_flags);
    bool ok;
};

const Api& api() {
    static const Api a = [] {
        Api x{};
        x.ok = resolve("cuMemCreate", &x.create) && resolve("cuMemRelease", &x.release) &&
               resolve("cuMemExportToShareableHandle", &x.exportH) && resolve("cuMemImportFromShareableHandle", &x.importH) &&
               resolve("cuMemAddressReserve", &x.reserve) && resolve("cuMemAddressFree", &x.addrFree) &&
               resolve("cuMemMap", &x.map) && resolve("cuMemUnmap", &x.unmap) && resolve("cuMemSetAccess", &x.setAccess) &&
               resolve("cuMemGetAllocationGranularity", &x.granularity);
        return x;
    }();
    return a;
}

CUmemAllocationProp props(int device) {
    CUmemAllocationProp p{};
    p.type = CU_MEM_ALLOCATION_TYPE_PINNED;
    p.location.type = CU_MEM_LOCATION_TYPE_DEVICE;
    p.location.id = device;
    p.requestedHandleTypes = CU_MEM_HANDLE_TYPE_POSIX_FILE_DESCRIPTOR;
    return p;
}

}  // namespace

extern "C" {

size_t fft3d_vmm_granularity(void) {
    int dev = 0;
    if (!api().ok || cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return 0; }
    cudaFree(nullptr);                                   // make sure the primary context exists
    const CUmemAllocationProp p = props(dev);
    size_t g = 0;
    if (api().granularity(&g, &p, CU_MEM_ALLOC_GRANULARITY_RECOMMENDED) != CUDA_SUCCESS) return 0;
    return g;
}

int fft3d_vmm_create(size_t bytes, unsigned long long* handle_out, int* fd_out) {
    if (handle_out == nullptr || bytes == 0) return FFT3D_EINVAL;
    int dev = 0;
    if (!api().ok || cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return FFT3D_ECUDA; }
    cudaFree(nullptr);
    const size_t g = fft3d_vmm_granularity();
    if (g == 0 || bytes % g != 0) return FFT3D_EINVAL;
    const CUmemAllocationProp p = props(dev);
    CUmemGenericAllocationHandle h = 0;
    if (api().create(&h, bytes, &p, 0) != CUDA_SUCCESS) return FFT3D_ENOMEM;
    if (fd_out != nullptr) {
        int fd = -1;
        if (api().exportH(&fd, h, CU_MEM_HANDLE_TYPE_POSIX_FILE_DESCRIPTOR, 0) != CUDA_SUCCESS) { api().release(h); return FFT3D_ECUDA; }
        *fd_out = fd;
    }
    *handle_out = (unsigned long long)h;
    return FFT3D_OK;
}

int fft3d_vmm_import(int fd, unsigned long long* handle_out) {
    if (handle_out == nullptr || fd < 0) return FFT3D_EINVAL;
    if (!api().ok) return FFT3D_ECUDA;
    cudaFree(nullptr);
    CUmemGenericAllocationHandle h = 0;
    if (api().importH(&h, (void*)(uintptr_t)fd, CU_MEM_HANDLE_TYPE_POSIX_FILE_DESCRIPTOR) != CUDA_SUCCESS) return FFT3D_ECUDA;
    *handle_out = (unsigned long long)h;
    return FFT3D_OK;
}

int fft3d_vmm_map(const unsigned long long* handles, int n, size_t part_bytes, void** va_out) {
    if (handles == nullptr || va_out == nullptr || n < 1 || part_bytes == 0) return FFT3D_EINVAL;
    *va_out = nullptr;
    int dev = 0;
    if (!api().ok || cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return FFT3D_ECUDA; }
    const size_t g = fft3d_vmm_granularity();
    if (g == 0 || part_bytes % g != 0) return FFT3D_EINVAL;
    CUdeviceptr base = 0;
    const size_t total = part_bytes * (size_t)n;
    if (api().reserve(&base, total, g, 0, 0) != CUDA_SUCCESS) return FFT3D_ENOMEM;
    int mapped = 0;
    bool ok = true;
    for (; mapped < n && ok; ++mapped)
        ok = api().map(base + (size_t)mapped * part_bytes, part_bytes, 0, (CUmemGenericAllocationHandle)handles[mapped], 0) == CUDA_SUCCESS;
    if (!ok) --mapped;                                   // the failing one is not mapped
    if (ok) {
        CUmemAccessDesc acc{};
        acc.location.type = CU_MEM_LOCATION_TYPE_DEVICE;
        acc.location.id = dev;
        acc.flags = CU_MEM_ACCESS_FLAGS_PROT_READWRITE;
        ok = api().setAccess(base, total, &acc, 1) == CUDA_SUCCESS;
    }
    if (!ok) {
        for (int i = 0; i < mapped; ++i) api().unmap(base + (size_t)i * part_bytes, part_bytes);
        api().addrFree(base, total);
        return FFT3D_ECUDA;
    }
    *va_out = (void*)base;
    return FFT3D_OK;
}

int fft3d_vmm_unmap(void* va, int n, size_t part_bytes) {
    if (va == nullptr || n < 1 || !api().ok) return FFT3D_EINVAL;
    const CUdeviceptr base = (CUdeviceptr)va;
    bool ok = true;
    for (int i = 0; i < n; ++i) ok = (api().unmap(base + (size_t)i * part_bytes, part_bytes) == CUDA_SUCCESS) && ok;
    ok = (api().addrFree(base, part_bytes * (size_t)n) == CUDA_SUCCESS) && ok;
    return ok ? FFT3D_OK : FFT3D_ECUDA;
}

int fft3d_vmm_release(unsigned long long handle) {
    if (!api().ok) return FFT3D_ECUDA;
    return api().release((CUmemGenericAllocationHandle)handle) == CUDA_SUCCESS ? FFT3D_OK : FFT3D_ECUDA;
}

}  // extern "C"
